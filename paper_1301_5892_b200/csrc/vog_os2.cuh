// vog_os2.cuh -- overlap-save advection kernels (line length N >= 1024).
// Product code; shares nothing with oracle/.
//
// The circulant product of P:98-100 taken block-wise in Fourier space: blocks of LB = 256 samples of the
// rolled line, V kept, H_lo discarded on the left (geometry (V, H_lo) = (232, 8) for Lagrange plans, (228, 14) for the
// cubic spline; template parameters).  The interpolation matrix is REAL, so two blocks A, B of the SAME line share the
// symbol lambda and ride one complex transform:  z_n = A_n + i B_n,  Z = FFT_256(z),  Z_k *= lambda_k
// (lambda_{256-k} = conj lambda_k),  z' = IFFT(Z)  =>  A' = Re z', B' = Im z'.  A work item is ONE radix-16 butterfly
// (16 complex = 32 registers) in every phase:
//   pass A   : item (pair, t):  n = t + 16 k  -> radix 16 over k, times W_256^{t k1}, stored at [k1][t]
//   middle   : item (pair, g = k1): radix 16 over t -> Z_{g + 16 k2}; times lambda; inverse radix 16
//   inverse A: item (pair, j): times conj W, inverse radix 16 over k1 -> z'_{j + 16 m}; the kept samples of both
//              blocks go straight to global memory.
// Every phase has 16 items per pair and every item touches only its own 16 scratch slots.  The full integer shift b of
// P:107 is applied by addressing.  Kernels in this file: osx7_kernel (x, default: per-pair windows landed by bulk
// copies), osx6_kernel (x, whole lines landed by bulk copies; 16384-cell lines), osv7_kernel (v, default: 16-column
// strips, three groups per CTA, raw rows by 2-D tensor copies), osv6_kernel / osv4_kernel (v fallbacks).
#pragma once
#include <cuda.h>

#include "vog_fft.cuh"
#include "vog_internal.h"

namespace vog {

// (working builds only, -DVOG_STAMPS: globaltimer stamps of the phases of CTA 0, read with vog_debug_os_stamps)
#ifdef VOG_STAMPS
__device__ long long os_stamps[64];
#define OS_STAMP(i) do { if (blockIdx.x == 0 && threadIdx.x == 0) { long long t_; asm volatile("mov.u64 %0, %%globaltimer;" : "=l"(t_)); os_stamps[i] = t_; } } while (0)
__device__ long long os_blk[4 * 1024];
#define OS_BLK(i) do { if (threadIdx.x == 0 && blockIdx.x < 1024) { long long t_; asm volatile("mov.u64 %0, %%globaltimer;" : "=l"(t_)); os_blk[4 * blockIdx.x + (i)] = t_; } } while (0)
#else
#define OS_STAMP(i) do { } while (0)
#define OS_BLK(i) do { } while (0)
#endif

namespace os2 {

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

// ---------------------------------------------------------------------------------------------
// mbarrier helpers (shared::cta)
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
// ---------------------------------------------------------------------------------------------
// x-direction, bulk-landed variant (default).  A persistent CTA owns whole lines.  ONE elected thread copies the next
// line group -- each line, the first XPAD cells of the line again behind its tail, and the line's symbol-table row --
// into shared memory with bulk asynchronous copies (cp.async.bulk, the TMA engine; completion is counted in bytes on an
// mbarrier), so no warp ever waits on its own global loads and no load occupies registers across its latency:
//   * pass A reads its samples n = t + 16 k from the line in shared memory, the integer shift b of P:107 applied by
//     addressing (4-byte loads, 16 consecutive words per half-warp: conflict free); the repeated head makes the
//     window of every item contiguous, so there is no wrap-around branch and no index masking per sample;
//   * the line buffer is free again once every warp has its samples in registers: each warp bumps a shared counter
//     after its (last) pass A, and the warp that completes the count issues the copies of the CTA's next line group,
//     which then land during the middle stage and the inverse pass (and under the other CTAs of the SM);
//   * in place needs no barrier at all: a line is completely on chip before the first store to it is issued.
// The phases of a pair are warp-private (the 16 items of a pair are 16 consecutive lanes in every phase: __syncwarp only).
// The symbol rows are double-buffered (2 x 1040 B per line): slow warps may still be in the middle stage of group g
// when the rows of group g+1 arrive.
namespace os2 {
constexpr int XPAD = 480;              // >= 240 + V + 1: the last sample of an item's window is c0 + 240 + V

__device__ __forceinline__ void mbar_expect_tx(unsigned long long* bar, const unsigned bytes)
{
    const unsigned s = (unsigned)__cvta_generic_to_shared(bar);
    asm volatile("mbarrier.arrive.expect_tx.shared::cta.b64 _, [%0], %1;\n" ::"r"(s), "r"(bytes) : "memory");
}
// global -> shared bulk copy (16-byte aligned addresses, size a multiple of 16), completing on bar
__device__ __forceinline__ void bulk_g2s(void* smem, const void* gmem, const unsigned bytes, unsigned long long* bar)
{
    const unsigned d = (unsigned)__cvta_generic_to_shared(smem), b = (unsigned)__cvta_generic_to_shared(bar);
    asm volatile("cp.async.bulk.shared::cluster.global.mbarrier::complete_tx::bytes [%0], [%1], %2, [%3];\n" ::"r"(d),
                 "l"(gmem), "r"(bytes), "r"(b)
                 : "memory");
}
__device__ __forceinline__ void mbar_init_fence() { asm volatile("fence.mbarrier_init.release.cluster;\n" ::: "memory"); }
// request a global range into L2 (no destination on chip, nothing to wait for)
__device__ __forceinline__ void bulk_prefetch_l2(const void* gmem, const unsigned bytes)
{
    asm volatile("cp.async.bulk.prefetch.L2.global [%0], %1;\n" ::"l"(gmem), "r"(bytes) : "memory");
}
}  // namespace os2

// kept samples of a FULL pair (both blocks inside the line): no bounds predicates, only the per-thread one of the
// partially kept sample row (m = 0 with the Lagrange geometry)
template <int V, int HLO, int M = 0>
__device__ __forceinline__ void os2_store_x_full(float* __restrict__ o, const int t, const float2* x)
{
    if constexpr (M < 16) {
        using K = KeptM<V, HLO, M>;
        if constexpr (K::all) {
            __stcs(o + 16 * M, x[M].x);
            __stcs(o + 16 * M + V, x[M].y);
        } else if constexpr (!K::none) {
            if (K::kept(t)) {
                __stcs(o + 16 * M, x[M].x);
                __stcs(o + 16 * M + V, x[M].y);
            }
        }
        os2_store_x_full<V, HLO, M + 1>(o, t, x);
    }
}

// LPI = 2: two lines per group as a compile-time constant AND one round with every thread busy (32 np == blockDim.x: the
// host checks it); LPI = 0: everything at run time (one line per group at 8192 cells, two rounds per group at 16384).
template <int V, int HLO, int LPI = 0>
__global__ void __launch_bounds__(288, 3) osx6_kernel(const OsArgs a)
{
    extern __shared__ __align__(128) unsigned char smem_raw[];
    const int lpi = LPI ? LPI : a.lpi, np = a.np, nitem = LPI ? (int)blockDim.x : lpi * np * 16;
    const int tid = threadIdx.x, T = blockDim.x, t = tid & 15;
    const int N = a.N, mask = N - 1, LS = N + os2::XPAD;
    float* const lines = reinterpret_cast<float*>(smem_raw);                       // lpi lines of LS floats
    float2* const lamS = reinterpret_cast<float2*>(lines + lpi * LS);              // [2][lpi][OS_LAMW]
    float2* const scr = lamS + 2 * lpi * OS_LAMW;                                  // (T / 16) pairs
    unsigned long long* const bar = reinterpret_cast<unsigned long long*>(scr + (T >> 4) * os2::XPAIR);   // [0] full, [1] empty
    Tw4 w;
    w.b1 = __ldg(a.tw + t);               // [q-1][t] = e^{-2 pi i t q / 256}
    w.b2 = __ldg(a.tw + 16 + t);
    w.b4 = __ldg(a.tw + 3 * 16 + t);
    w.b8 = __ldg(a.tw + 7 * 16 + t);
    if (tid == 0) {
        os2::mbar_init(bar, 1);                   // full: the elected thread's expect_tx arrival + the bytes of the copies
        os2::mbar_init(bar + 1, T >> 5);          // empty: one arrival per warp, after its last pass A of the group
        os2::mbar_init_fence();
    }
    __syncthreads();
    pdl_wait();                                   // (the twiddles above are plan constants; tables and grid are not)
    pdl_launch_dependents();
    // copies of line group g into the line buffers and into symbol-row buffer (par); called by ONE thread.  The lines of
    // the group after it are requested into L2 at the same time: their HBM latency (and the queueing behind everyone
    // else's requests) then runs two groups ahead and costs no shared memory; the copy proper is an L2 hit.
    auto issue = [&](const int g, const unsigned par) {
        const int line0 = g * lpi, nl = min(lpi, a.n_lines - line0);
        os2::mbar_expect_tx(bar, (unsigned)nl * (unsigned)(4 * LS + 8 * OS_LAMW));
        for (int l = 0; l < nl; ++l) {
            const float* gl = a.src + (size_t)(line0 + l) * N;
            os2::bulk_g2s(lines + l * LS, gl, 4u * (unsigned)N, bar);
            os2::bulk_g2s(lines + l * LS + N, gl, 4u * os2::XPAD, bar);
            os2::bulk_g2s(lamS + (par * lpi + l) * OS_LAMW, a.lam + (size_t)(line0 + l) * OS_LAMW, 8u * OS_LAMW, bar);
        }
        const int line2 = (g + (int)gridDim.x) * lpi, nl2 = min(lpi, a.n_lines - line2);
        for (int l = 0; l < nl2; ++l) os2::bulk_prefetch_l2(a.src + (size_t)(line2 + l) * N, 4u * (unsigned)N);
    };
    if (tid == 0 && (int)blockIdx.x < a.n_groups) issue(blockIdx.x, 0u);
    float2* const sA = scr + (tid >> 4) * os2::XPAIR + t;                          // passes A: column t of the pair
    float2* const sM = scr + (tid >> 4) * os2::XPAIR + os2::XROW * t;              // middle stage: row g = t
    unsigned parity = 0;
    for (int g = blockIdx.x; g < a.n_groups; g += gridDim.x) {
        os2::mbar_wait(bar, parity);              // the lines and symbol rows of this group have landed
        const float2* const lamG = lamS + parity * lpi * OS_LAMW;
        const int gn = g + gridDim.x;
#pragma unroll 1
        for (int it0 = 0; it0 < nitem; it0 += T) {                      // rounds (one when the group fits the CTA)
            const int it = it0 + tid;
            const bool active = LPI ? true : it < nitem;
            const int pr = it >> 4;
            const int l = LPI == 2 ? (pr >= np ? 1 : 0) : (int)(((unsigned)pr * a.inv_np) >> 16);
            const int pp = pr - l * np;                                               // line of the group, pair of the line
            const float2* const lamL = lamG + l * OS_LAMW;
            // ---- pass A from the line in shared memory
            if (active) {
                const int b = __float_as_int(lamL[129].x);
                const float* const p = lines + l * LS + ((pp * (2 * V) - HLO + b + t) & mask);
                float2 x[16];
#pragma unroll
                for (int k = 0; k < 16; ++k) x[k] = make_float2(p[16 * k], p[16 * k + V]);
                dft_dif<16, 1>(x);
                sA[0] = x[0];
                os2_tw_each(w, [&](auto qc, const float2 y) {
                    constexpr int q = decltype(qc)::value;
                    sA[os2::XROW * q] = cmul(x[brev(q, 16)], y);
                });
            }
            __syncwarp();
            // (the shared stores above needed every sample: this warp is done with the line buffers)
            const bool last_round = it0 + T >= nitem;
            if (last_round && (tid & 31) == 0) os2::mbar_arrive(bar + 1);
            // ---- middle stage
            if (active) {
                float2 x[16];
#pragma unroll
                for (int j = 0; j < 16; ++j) x[j] = sM[j];
                os2::mid16<1>(x, lamL, t);
#pragma unroll
                for (int j = 0; j < 16; ++j) sM[j] = x[j];
            }
            // once every warp is done with the line buffers, thread 0 requests the CTA's next line group; it lands
            // behind the inverse pass (by now the other warps have normally arrived: the wait is a formality)
            if (last_round && tid == 0 && gn < a.n_groups) {
                os2::mbar_wait(bar + 1, parity);
                issue(gn, parity ^ 1u);
            }
            __syncwarp();
            // ---- inverse pass A: scratch -> registers -> global
            if (active) {
                float2 x[16];
                x[0] = sA[0];
                os2_tw_each(w, [&](auto qc, const float2 y) {
                    constexpr int q = decltype(qc)::value;
                    x[brev(q, 16)] = cmulc(sA[os2::XROW * q], y);
                });
                idft_dit<16, 1>(x);
                const int line = g * lpi + l;
                if (line < a.n_lines) {
                    const int c = pp * (2 * V) + t - HLO;          // cell of sample n = t of block A
                    float* const o = a.dst + (size_t)line * N + c;
                    if ((pp + 1) * (2 * V) <= N) os2_store_x_full<V, HLO>(o, t, x);
                    else os2_store_x<V, HLO>(o, c, N, t, false, x);
                }
            }
            __syncwarp();                          // the scratch of this warp is rewritten by its next pass A
        }
        parity ^= 1u;
    }
}

// ---------------------------------------------------------------------------------------------
// x-direction, warp-private windows (default when a line group fits one round of the CTA, i.e. lines up to 8192 cells).
// osx6_kernel lands whole lines for the whole CTA, so every warp waits for the slowest one twice per line (the line
// buffer must be empty before it is refilled, and full before anybody starts): measured, a quarter of all warp time
// sat in that wait.  Here each half-warp copies exactly the WINDOW of its own pair -- 256 + V consecutive cells of the
// rolled line, 16-byte aligned, at most two bulk copies when it wraps around the end of the line -- into its own 2 KB
// slot, counted on its WARP's mbarrier:
//   * a warp refills its slots as soon as ITS pass A is done and waits only for ITS windows: loads, transforms and
//     stores of different warps overlap freely, as in the register-landing kernel, but nobody waits on a global load;
//   * in place: a store to line g may only be issued once every window of line g is on chip.  Each warp arrives on a
//     CTA-wide "landed" mbarrier when it has seen its windows and checks it before its first store, two phases later
//     (pass A and the middle stage lie in between), so the check practically never blocks;
//   * the integer shift b of the NEXT group's line is fetched one iteration ahead, the lines of the group after next are
//     requested into L2, and the symbol row (1 KB per line, shared by the warps of the line) is read through L1.
// Slots of 496 floats put the two windows of a warp 16 banks apart for either block geometry: pass A is conflict free.
namespace os2 {
constexpr int XWIN = 492;              // floats per window slot = floats copied per window: 3 (alignment) + 15 + 240 + V + 1
constexpr int XCOPY = XWIN;
}

template <int V, int HLO>
__global__ void __launch_bounds__(288, 3) osx7_kernel(const OsArgs a)
{
    extern __shared__ __align__(128) unsigned char smem_raw[];
    const int lpi = a.lpi, np = a.np, nitem = lpi * np * 16;        // nitem <= blockDim.x: one item per thread and phase
    const int tid = threadIdx.x, T = blockDim.x, t = tid & 15, hw = tid >> 4, lane = tid & 31, warp = tid >> 5;
    const int N = a.N, mask = N - 1, nwarps = T >> 5;
    // shared memory (sized to the byte: three CTAs of 18 pairs fill an SM): window slots | symbol rows [2][lpi] | exchange
    // scratch (the unused last pad element of a pair's 16 x 17 block overlaps the next pair's first) | shifts | mbarriers
    const int S = T >> 4;                                                                          // pair slots
    float* const win = reinterpret_cast<float*>(smem_raw) + hw * os2::XWIN;                       // this pair's window
    float2* const lamS = reinterpret_cast<float2*>(reinterpret_cast<float*>(smem_raw) + S * os2::XWIN);   // [2][lpi][OS_LAMW]
    float2* const scr = lamS + 2 * lpi * OS_LAMW + hw * (os2::XPAIR - 1);
    int* const wsh = reinterpret_cast<int*>(lamS + 2 * lpi * OS_LAMW + S * (os2::XPAIR - 1) + 1) + 2 * hw;   // [S][2]
    unsigned long long* const bars = reinterpret_cast<unsigned long long*>(
        reinterpret_cast<int*>(lamS + 2 * lpi * OS_LAMW + S * (os2::XPAIR - 1) + 1) + 2 * S);
    // bars: [0] landed; [1] symbol rows; [2 + warp] windows of the warp
    Tw4 w;
    w.b1 = __ldg(a.tw + t);               // [q-1][t] = e^{-2 pi i t q / 256}
    w.b2 = __ldg(a.tw + 16 + t);
    w.b4 = __ldg(a.tw + 3 * 16 + t);
    w.b8 = __ldg(a.tw + 7 * 16 + t);
    // (one barrier per thread: a loop over the barriers in ONE thread made ptxas 12.9 read the uniform register that
    // holds the address of the last barrier before writing it, and the kernel then waited on an uninitialised object)
    if (tid <= nwarps + 1) {
        // [0]: one arrival per warp; [1]: thread 0's expect_tx; others: the two half-warp leaders' expect_tx arrivals
        os2::mbar_init(bars + tid, tid == 0 ? (unsigned)nwarps : (tid == 1 ? 1u : 2u));
        os2::mbar_init_fence();
    }
    __syncthreads();
    pdl_wait();                                   // (the twiddles above are plan constants; tables and grid are not)
    pdl_launch_dependents();
    const bool has_pair = hw * 16 < nitem;
    const int l = (int)(((unsigned)hw * a.inv_np) >> 16), pp = hw - l * np;    // line of the group, pair of the line
    const int G = gridDim.x;
    float2* const sA = scr + t;                                                // passes A: column t of the pair
    float2* const sM = scr + os2::XROW * t;                                    // middle stage: row g = t
    // leader of a half-warp (t == 0): request this pair's window of line group g, whose line has the integer shift b
    auto issue = [&](const int g, const int b) {
        const int line = g * lpi + l;
        if (!has_pair || line >= a.n_lines) { os2::mbar_arrive(bars + 2 + warp); return; }
        os2::mbar_expect_tx(bars + 2 + warp, 4u * os2::XCOPY);
        const float* const gl = a.src + (size_t)line * N;
        const int a0 = ((pp * (2 * V) - HLO + b) & mask) & ~3;
        if (a0 + os2::XCOPY <= N) os2::bulk_g2s(win, gl + a0, 4u * os2::XCOPY, bars + 2 + warp);
        else {
            const int n1 = N - a0;
            os2::bulk_g2s(win, gl + a0, 4u * (unsigned)n1, bars + 2 + warp);
            os2::bulk_g2s(win + n1, gl, 4u * (unsigned)(os2::XCOPY - n1), bars + 2 + warp);
        }
    };
    // The integer shifts travel through two words of shared memory per pair, so that no register holds them across
    // a phase (they were spilled, and the spill waited for the load): wsh[1] = shift of the window in flight (written
    // by the leader when it requests the window, read by the 16 threads in pass A), wsh[0] = shift of the group after
    // that, fetched by a 4-byte cp.async one iteration ahead.
    auto fetch_shift = [&](const int g) {          // leader: shift of this pair's line in group g -> wsh[0], asynchronously
        const int line = g * lpi + l;
        if (has_pair && g < a.n_groups && line < a.n_lines) os2::cp_async4(wsh, &a.lam[(size_t)line * OS_LAMW + 129].x);
    };
    // thread 0: symbol rows of the lines of group g into row buffer (par).  Called for group g + G right after the
    // landed barrier of group g: by then every warp has started pass A of group g, i.e. is done with the middle stage
    // of group g - G, whose rows this overwrites; they arrive long before the first middle stage of group g + G.
    auto issue_rows = [&](const int g, const unsigned par) {
        const int line0 = g * lpi, nl = min(lpi, a.n_lines - line0);
        os2::mbar_expect_tx(bars + 1, (unsigned)nl * 8u * OS_LAMW);
        for (int i = 0; i < nl; ++i)
            os2::bulk_g2s(lamS + (par * lpi + i) * OS_LAMW, a.lam + (size_t)(line0 + i) * OS_LAMW, 8u * OS_LAMW, bars + 1);
    };
    if ((int)blockIdx.x < a.n_groups) {
        if (t == 0) {
            const int line = blockIdx.x * lpi + l;
            const int b0 = (has_pair && line < a.n_lines) ? __float_as_int(__ldg(&a.lam[(size_t)line * OS_LAMW + 129].x)) : 0;
            wsh[1] = b0;
            issue(blockIdx.x, b0);
            fetch_shift(blockIdx.x + G);
        }
        if (tid == 0) issue_rows(blockIdx.x, 0u);
    }
    unsigned parity = 0;
    for (int g = blockIdx.x; g < a.n_groups; g += G) {
        const int gn = g + G;
        const int line = g * lpi + l;
        const bool active = has_pair && line < a.n_lines;
        os2::mbar_wait(bars + 2 + warp, parity);   // this warp's windows have landed
        // (the symbol rows of this group were requested a whole group ago.  The wait sits HERE, before the arrival on
        // the landed barrier, because thread 0 re-arms the row barrier right after the landed barrier completes: a
        // warp that had not yet observed this phase would then miss it and wait for ever.)
        os2::mbar_wait(bars + 1, parity);
        if (lane == 0) os2::mbar_arrive(bars);
        // ---- pass A from the window
        if (active) {
            const int b = wsh[1];
            const float* const p = win + (((pp * (2 * V) - HLO + b) & mask) & 3) + t;
            float2 x[16];
#pragma unroll
            for (int k = 0; k < 16; ++k) x[k] = make_float2(p[16 * k], p[16 * k + V]);
            dft_dif<16, 1>(x);
            sA[0] = x[0];
            os2_tw_each(w, [&](auto qc, const float2 y) {
                constexpr int q = decltype(qc)::value;
                sA[os2::XROW * q] = cmul(x[brev(q, 16)], y);
            });
        }
        __syncwarp();
        // (the shared stores above needed every sample: the window slots of this warp are free)
        if (gn < a.n_groups) {
            if (t == 0) {
                os2::cp_async_wait_all();          // the shift fetched one iteration ago
                const int bn = wsh[0];
                wsh[1] = bn;
                issue(gn, bn);
                fetch_shift(gn + G);
                if (pp == 0 && has_pair && (gn + G) * lpi + l < a.n_lines)
                    os2::bulk_prefetch_l2(a.src + (size_t)((gn + G) * lpi + l) * N, 4u * (unsigned)N);
            }
        }
        // ---- middle stage
        if (active) {
            float2 x[16];
#pragma unroll
            for (int j = 0; j < 16; ++j) x[j] = sM[j];
            os2::mid16<1>(x, lamS + (parity * lpi + l) * OS_LAMW, t);
#pragma unroll
            for (int j = 0; j < 16; ++j) sM[j] = x[j];
        }
        __syncwarp();
        os2::mbar_wait(bars, parity);              // every window of this line group is on chip: stores may begin
        if (tid == 0 && gn < a.n_groups) issue_rows(gn, parity ^ 1u);
        // ---- inverse pass A: scratch -> registers -> global
        if (active) {
            float2 x[16];
            x[0] = sA[0];
            os2_tw_each(w, [&](auto qc, const float2 y) {
                constexpr int q = decltype(qc)::value;
                x[brev(q, 16)] = cmulc(sA[os2::XROW * q], y);
            });
            idft_dit<16, 1>(x);
            const int c = pp * (2 * V) + t - HLO;          // cell of sample n = t of block A
            float* const o = a.dst + (size_t)line * N + c;
            if ((pp + 1) * (2 * V) <= N) os2_store_x_full<V, HLO>(o, t, x);
            else os2_store_x<V, HLO>(o, c, N, t, false, x);
        }
        __syncwarp();                              // the scratch of this warp is rewritten by its next pass A
        parity ^= 1u;
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
// delta-f source on the samples of one item: x[m].x += f_eq,g(v_j)(e^{X_j} - 1) at rows j = r0 + 16 m
// (r0 = row of sample n = t of block A), x[m].y the same at rows j + V, with X_j = c s (2 (v_j - mu) - s) affine in j.
// Along rows 16 apart expm1 obeys e' = e R + r (R = e^h, r = expm1(h), h = 32 c s dv); the recurrence starts in
// the middle (m = 8) and runs both ways (RS[g] = (R, r, 1/R, expm1(-h)) per lane), so at most 8 steps accumulate.
// Sample rows without kept samples (m = 15 and/or m = 0, depending on the geometry) are skipped.  The f_eq table
// has 512 floats of padding: rows >= Nv are read but never stored; rows < 0 (m = 0 of the first pair) are clamped.
template <int V, int HLO, int W = 32>
__device__ __forceinline__ void osv2_source(float2* x, const OsArgs& a, const float4* __restrict__ RS, const int lane,
                                            const int r0, const float ssh, const float2* __restrict__ RV = nullptr)
{
    constexpr int M0 = KeptM<V, HLO, 0>::none ? 1 : 0;       // first and last sample rows that hold kept samples
    constexpr int M1 = KeptM<V, HLO, 15>::none ? 14 : 15;
#pragma unroll 1
    for (int g = 0; g < a.ng; ++g) {
        const float cgs = a.cg4[g] * ssh;
        const float* __restrict__ fa = a.feq_tab + g * a.Nv + r0;
        const float u0 = __ldg(a.vmu_tab + g * a.Nv);                          // v_0 - mu_g
        float4 Rr;
        if (RS) Rr = RS[g * W + lane];
        else {                                   // (the 16-column kernel has no room for the table)
            const float hh = 32.0f * cgs * a.dvf;
            Rr = make_float4(expf(hh), expm1f(hh), expf(-hh), expm1f(-hh));
        }
        const float ea8 = expm1f(cgs * (2.0f * fmaf((float)(r0 + 128), a.dvf, u0) - ssh));
        // (block B lies V rows further: e^{X + g V} - 1 = (e^X - 1) e^{g V} + (e^{g V} - 1), RV = (e^{g V}, expm1(g V)) per lane)
        float eb8;
        if (RV) { const float2 rv = RV[g * W + lane]; eb8 = fmaf(ea8, rv.x, rv.y); }
        else eb8 = expm1f(cgs * (2.0f * fmaf((float)(r0 + 128 + V), a.dvf, u0) - ssh));
        float ea = ea8, eb = eb8;
#pragma unroll
        for (int m = 8; m <= M1; ++m) {
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
    extern __shared__ __align__(128) unsigned char smem_raw[];
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
            os2::cp_async16(dst4 + i, src4 + (size_t)(i >> 4) * (a.lam_ks / 2) + (i & 15));
    }
    // integer shift (rows) and source shift of this lane's column
    const float2 e129 = __ldg(a.lam + (size_t)129 * a.lam_ks + c0 + lane);
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


// ---------------------------------------------------------------------------------------------
// v-direction, 16-column strips with the next window in flight (default).  Same arithmetic as osv4_kernel, other
// shape: a strip is 16 adjacent columns (64-byte row segments), an item (t, g or j) is a HALF-warp, a CTA is 8 warps
// and handles one pair of blocks of its strip per iteration.  The raw rows (the union of the rows the 16 columns need,
// landed unshifted by 16-byte cp.async) and the exchange buffer are SEPARATE 32 KB buffers, so
//   * the raw rows of the CTA's NEXT pair are requested as soon as pass A has emptied the raw buffer and land during
//     the middle stage and the inverse pass (the 32-column kernel shares one buffer and loads nothing while it computes);
//   * three CTA barriers per pair instead of five;
//   * 64 KB per CTA: three CTAs (24 warps) per SM, out of phase with one another.
// The symbol table of the strip is read straight from global memory ([k][column]: a half-warp reads one 128-byte
// row; 16.5 KB per strip, re-read for every pair, so it lives in L1 -- f itself is loaded with cp.async.cg, which
// bypasses L1).  Bank conflicts: raw[row][16] floats -- a lane only touches bank (column + 16 (row & 1)), and the two
// half-warps of a warp read rows of opposite parity (items t, t + 1): conflict free for any per-column shift;
// exchange [position][16] float2 -- a half-warp covers one 128-byte row: conflict free.
// Strips whose integer shifts spread over more rows than the raw buffer holds fall back to a per-lane landing of the
// same buffer (4-byte cp.async).  Out of place (src != dst).
namespace os2 {
__device__ __forceinline__ void cp_async16_cg(void* smem, const void* gmem)
{
    const unsigned s = (unsigned)__cvta_generic_to_shared(smem);
    asm volatile("cp.async.cg.shared.global [%0], [%1], 16;\n" ::"r"(s), "l"(gmem) : "memory");
}
constexpr int VW = 16;                 // columns per strip
constexpr int VRR = 516;               // rows of the raw buffer (33 KB + 32 KB of exchange buffer: three CTAs per SM
                                       // inside the 196 KB shared-memory carve-out, which leaves ~60 KB of L1 for the
                                       // symbol tables of the three strips)
}  // namespace os2

// kept samples of a FULL pair along rows (row stride Nx): no bounds predicates
template <int V, int HLO, int M = 0>
__device__ __forceinline__ void os2_store_v_full(float* __restrict__ po, const size_t Nx, const int t, const float2* x)
{
    if constexpr (M < 16) {
        using K = KeptM<V, HLO, M>;
        if constexpr (K::all) {
            __stcs(po + (size_t)(16 * M) * Nx, x[M].x);
            __stcs(po + (size_t)(16 * M + V) * Nx, x[M].y);
        } else if constexpr (!K::none) {
            if (K::kept(t)) {
                __stcs(po + (size_t)(16 * M) * Nx, x[M].x);
                __stcs(po + (size_t)(16 * M + V) * Nx, x[M].y);
            }
        }
        os2_store_v_full<V, HLO, M + 1>(po, Nx, t, x);
    }
}

template <int V, int HLO>
__global__ void __launch_bounds__(256, 3) osv6_kernel(const OsArgs a)
{
    extern __shared__ __align__(128) unsigned char smem_raw[];
    constexpr int W = os2::VW, RR = os2::VRR;
    constexpr int RMAX = RR - OS_LB - V;           // spread of the integer shifts that the raw buffer can hold
    float* const raw = reinterpret_cast<float*>(smem_raw);                        // [RR][16]
    float2* const exch = reinterpret_cast<float2*>(raw + RR * W);                 // [256][16]
    const int tid = threadIdx.x, c = tid & 15, h = tid >> 4;                      // column of the strip, item index
    const int Nx = a.Nx, Nv = a.Nv, vmask = Nv - 1;
    const int c0 = blockIdx.x * W;
    Tw4 w;
    w.b1 = __ldg(a.tw + h);                       // [q-1][t] = e^{-2 pi i t q / 256}, t = item index of passes A
    w.b2 = __ldg(a.tw + 16 + h);
    w.b4 = __ldg(a.tw + 3 * 16 + h);
    w.b8 = __ldg(a.tw + 7 * 16 + h);
    pdl_wait();                                   // the symbol tables and the source grid come from earlier kernels
    pdl_launch_dependents();
    const float2* __restrict__ const lamC = a.lam + c0 + c;                       // entry k of this column: lamC[k ks]
    // integer shift (rows) and source shift of this lane's column
    const size_t ks = (size_t)a.lam_ks;            // row stride of the table: Nx + 16 entries (not a power of two: the 129
                                                  // rows of a strip fall into different L1 sets)
    const float2 e129 = __ldg(lamC + 129 * ks);
    const int b = __float_as_int(e129.x);
    const float ssh = e129.y;
    // spread of the shifts over the strip, as signed distances from column 0's (shifts live mod Nv)
    const int b0 = __shfl_sync(0xffffffffu, b, 0, 16);
    const int d = (((b - b0) + (Nv >> 1)) & vmask) - (Nv >> 1);
    int dmin = d, dmax = d;
#pragma unroll
    for (int o = 8; o > 0; o >>= 1) {
        dmin = min(dmin, __shfl_xor_sync(0xffffffffu, dmin, o));
        dmax = max(dmax, __shfl_xor_sync(0xffffffffu, dmax, o));
    }
    const int R = dmax - dmin;
    const bool gather = R > RMAX;                  // uniform over the CTA (every half-warp sees the same 16 columns)
    const int db = gather ? 0 : d - dmin;          // this lane's row offset inside the raw window
    const int base = gather ? b : b0 + dmin;       // first raw row = pair start - HLO + base
    const float* const col = a.src + c0 + c;
    float* const ocol = a.dst + c0 + c;
    const int p0 = blockIdx.y * a.gpc, p1 = min(a.np, p0 + a.gpc);
    float2* const own = exch + h * W + c;                                     // position t = h
    constexpr int PS = 16 * W;                                                // float2 between positions 16 apart
    const int nrows = V + OS_LB + (gather ? 0 : R);

    // request the raw rows of pair p: the union of the rows, unshifted (or, in the fallback, every lane its own rows)
    auto land = [&](const int p) {
        const int rs = p * (2 * V) - HLO + base;
        if (!gather) {
            const float* const src = a.src + c0;
            for (int i = tid; i < nrows * 4; i += 256) {
                const int r = i >> 2, q4 = (i & 3) * 4;
                os2::cp_async16_cg(raw + r * W + q4, src + (size_t)((rs + r) & vmask) * Nx + q4);
            }
        } else {
            for (int r = h; r < nrows; r += 16) os2::cp_async4(raw + r * W + c, col + (size_t)((rs + r) & vmask) * Nx);
        }
    };
    if (p0 < p1) land(p0);
    for (int p = p0; p < p1; ++p) {
        os2::cp_async_wait_all();
        __syncthreads();                           // raw rows of pair p visible; exchange buffer of pair p - 1 read
        // ---- pass A (item t = h): samples from the raw rows with this lane's offset
        {
            float2 x[16];
            const float* const rp = raw + (h + db) * W + c;
#pragma unroll
            for (int k = 0; k < 16; ++k) x[k] = make_float2(rp[16 * k * W], rp[(16 * k + V) * W]);
            dft_dif<16, 1>(x);
            own[0] = x[0];
            os2_tw_each(w, [&](auto qc, const float2 y) {
                constexpr int q = decltype(qc)::value;
                own[q * PS] = cmul(x[brev(q, 16)], y);
            });
        }
        __syncthreads();                           // exchange buffer complete; raw rows all read
        if (p + 1 < p1) land(p + 1);               // the next window lands behind the middle stage and the inverse pass
        // ---- middle stage (item g = h): positions 16 g + j; symbol from the table in global memory (L1)
        {
            float2* const sp = exch + h * 16 * W + c;
            float2 x[16];
#pragma unroll
            for (int j = 0; j < 16; ++j) x[j] = sp[j * W];
            dft_dif<16, 1>(x);
#pragma unroll
            for (int q = 0; q < 8; ++q) x[brev(q, 16)] = cmul(x[brev(q, 16)], __ldg(lamC + (size_t)(h + 16 * q) * ks));
#pragma unroll
            for (int q = 8; q < 16; ++q) x[brev(q, 16)] = cmulc(x[brev(q, 16)], __ldg(lamC + (size_t)(256 - 16 * q - h) * ks));
            idft_dit<16, 1>(x);
#pragma unroll
            for (int j = 0; j < 16; ++j) sp[j * W] = x[j];
        }
        __syncthreads();
        // ---- inverse pass A (item j = h): kept samples -> rows of the destination
        {
            float2 x[16];
            x[0] = own[0];
            os2_tw_each(w, [&](auto qc, const float2 y) {
                constexpr int q = decltype(qc)::value;
                x[brev(q, 16)] = cmulc(own[q * PS], y);
            });
            idft_dit<16, 1>(x);
            const int r0 = p * (2 * V) + h - HLO;          // row of sample n = t = h of block A
            if (a.ng > 0) osv2_source<V, HLO, W>(x, a, nullptr, c, r0, ssh);
            float* const po = ocol + (ptrdiff_t)r0 * Nx;
            if ((p + 1) * (2 * V) <= Nv) os2_store_v_full<V, HLO>(po, (size_t)Nx, h, x);
            else os2_store_v<V, HLO>(po, (size_t)Nx, r0, Nv, h, false, x);
        }
    }
}


// ---------------------------------------------------------------------------------------------
// v-direction, three groups per CTA sharing the strip's symbol table (default).  osv6_kernel reads the symbol through
// L1, and the profile shows that this is what it waits for (long-scoreboard stalls on the multiplies of the middle
// stage, L1 hit rate 18 %: three strips x 16.5 KB do not stay resident beside the streaming traffic).  Here ONE CTA of
// 768 threads per SM holds the table of its strip in shared memory (16.6 KB, staged once per work item) and runs
// THREE groups of 8 warps on it, each with its own raw-row buffer and exchange buffer (3 x 64.5 KB) and its own named
// barrier: the groups are the three CTAs of osv6_kernel, minus the table traffic, and drift apart in the same way.
// A work item is (strip of 16 columns, segment of consecutive pairs); group i takes pairs i, i + 3, .. of the segment
// and has the raw rows of its next pair in flight while it transforms the current one.  Persistent grid.
namespace os2 {
__device__ __forceinline__ void bar_group(const int id) { asm volatile("bar.sync %0, 256;\n" ::"r"(id) : "memory"); }
constexpr int VRT = 520;               // rows of a group's raw buffer in osv7_kernel (even: rows land two by two)
// tensor maps of the source grid [Nv][Nx] with boxes of 16 columns x {256, 64, 16, 4, 2} rows (host: osv7_launch)
struct VMaps { CUtensorMap m[5]; };
__device__ __forceinline__ int vbox_rows(const int i) { return i == 4 ? 2 : 256 >> (2 * i); }
// box (16 columns from column x, the map's rows from row y) -> shared memory (128-byte aligned), completing on bar
__device__ __forceinline__ void tensor_g2s(void* smem, const CUtensorMap* map, const int x, const int y,
                                           unsigned long long* bar)
{
    const unsigned d = (unsigned)__cvta_generic_to_shared(smem), b = (unsigned)__cvta_generic_to_shared(bar);
    asm volatile("cp.async.bulk.tensor.2d.shared::cluster.global.mbarrier::complete_tx::bytes [%0], [%1, {%2, %3}], [%4];\n"
                 ::"r"(d), "l"(reinterpret_cast<unsigned long long>(map)), "r"(x), "r"(y), "r"(b)
                 : "memory");
}
}

// Work of CTA kb of G in osv7_kernel, piece i: (strip of 16 columns, pairs q0 .. q1-1); false = no such piece.  The
// strips are dealt out round-robin in whole rounds of G strips (neighbouring CTAs work on neighbouring strips at the same
// time); the strips left over after the last whole round are cut by PAIRS into G equal shares, so every CTA gets the
// same number of pairs (+-1) whatever Nx / 16 is (8192: 512 strips on 148 CTAs were 4 rounds for 3.46 rounds of work).
__device__ __forceinline__ bool osv7_piece(const int i, const int G, const int kb, const int nstrips, const int np,
                                           int& strip, int& q0, int& q1)
{
    const int Rr = nstrips / G, Lt = nstrips - Rr * G;
    if (i < Rr) { strip = i * G + kb; q0 = 0; q1 = np; return true; }
    if (Rr == 0) {
        // fewer strips than CTAs (grids up to 2048 columns): a share of pairs would straddle two strips and pay two
        // tables for a handful of pairs; instead every strip gets floor(G / nstrips) CTAs, one segment each
        const int m = G / nstrips, sidx = kb / nstrips, sg = (np + m - 1) / m;
        strip = kb % nstrips;
        q0 = sidx * sg;
        q1 = min(np, q0 + sg);
        return i == 0 && sidx < m && q0 < q1;
    }
    const int tlo = (int)((long long)Lt * np * kb / G), thi = (int)((long long)Lt * np * (kb + 1) / G);
    int L = tlo;
    for (int j = i - Rr;; --j) {
        if (L >= thi) return false;
        const int sidx = L / np;
        q0 = L - sidx * np;
        q1 = min(np, q0 + thi - L);
        if (j == 0) { strip = Rr * G + sidx; return true; }
        L += q1 - q0;
    }
}

namespace os2 { constexpr int IPH = 40; }       // rows kept on either side of a piece of the in-place v kernel

// In-place v-advection, first launch (only when the v kernel's pieces are not all whole strips): the rows on either side
// of every such piece, which ANOTHER CTA of osv7_kernel will store, copied to a.halo [CTA][4][2][IPH][16] while the grid
// is still untouched.  Same grid as osv7_kernel (CTA kb saves for CTA kb of that launch), 256 threads.
static __global__ void __launch_bounds__(256) osv7_halo_kernel(const OsArgs a, const int V2)
{
    constexpr int W = os2::VW, IPH = os2::IPH;
    pdl_wait();                                   // the grid comes from the kernel before
    pdl_launch_dependents();
    const int G = gridDim.x, kb = blockIdx.x, np = a.np, vmask = a.Nv - 1;
    int s0, qa, qb, li = 0;
    for (int i = 0; li < 4 && osv7_piece(i, G, kb, a.Nx / W, np, s0, qa, qb); ++i) {
        if (qa == 0 && qb == np) continue;
        float* const hs = a.halo + (size_t)(kb * 4 + li) * (2 * IPH * W);
        const int lw = qa * V2, uw = qb < np ? qb * V2 : a.Nv;
        for (int j = threadIdx.x; j < 2 * IPH * W; j += 256) {
            const int side = j >= IPH * W, r = (j - side * IPH * W) >> 4, cc = j & (W - 1);
            const int row = (side ? uw + r : lw - IPH + r) & vmask;
            hs[j] = __ldcg(a.src + (size_t)row * a.Nx + s0 * W + cc);
        }
        ++li;
    }
}

// IPM = 0: out of place only, the in-place bookkeeping compiled out (grids of 4096 columns or more: with the run-time
// flag the out-of-place kernel was 2.3 % slower at 8192^2 than before the mode existed, 131.4 against 128.5 us; this
// instance takes 127.4 us); IPM = 2: a.inplace decides at run time (in-place calls, and the grids up to 2048 columns,
// where the compile-time instance made the 2048^2 step 2.1 us SLOWER: 46.15 -> 48.27 us, same box -- code generation
// of the prologue, not the flag).
template <int V, int HLO, int IPM = 2>
__global__ void __launch_bounds__(768, 1) osv7_kernel(const OsArgs a, const OsSetupArgs su,
                                                      const __grid_constant__ os2::VMaps maps)
{
    extern __shared__ __align__(128) unsigned char smem_raw[];
    constexpr int W = os2::VW, RR = os2::VRT;
    constexpr int RMAX = RR - OS_LB - V - 1;       // spread of the integer shifts that the raw buffer can hold (the
                                                   // window starts on an even row: up to one row more than needed)
    constexpr int GB = RR * W * 4 + OS_LB * W * 8; // bytes per group: raw rows + exchange buffer
    constexpr int CF = 20 * W;                     // words of one coefficient record: [18][16] floats, [16] b, [16] E dt
    constexpr int HEAD = OS_LAMW * W * 8 + 240 * 8 + 3 * CF * 4 + 136 * 16;   // a multiple of 128 bytes
    float2* const lamS = reinterpret_cast<float2*>(smem_raw);                     // [OS_LAMW][16]
    float2* const twS = lamS + OS_LAMW * W;                                       // [15][16] e^{-2 pi i t q / 256}
    float* const cfS = reinterpret_cast<float*>(twS + 240);                       // [3] coefficient records (ring)
    float4* const csS = reinterpret_cast<float4*>(cfS + 3 * CF);                  // [129] (cos, sin, ..) of theta_k
    const int tid = threadIdx.x, gid = tid >> 8, gt = tid & 255;                  // group, thread of the group
    unsigned char* const gbase = smem_raw + HEAD + gid * GB;
    float* const raw = reinterpret_cast<float*>(gbase);                           // [RR][16]
    float2* const exch = reinterpret_cast<float2*>(raw + RR * W);                 // [256][16]
    // one mbarrier per group: the bytes of the group's raw rows (one expect_tx arrival by the thread that requests them)
    unsigned long long* const vbar = reinterpret_cast<unsigned long long*>(smem_raw + HEAD + 3 * GB) + gid;
    unsigned vpar = 0;
    if (gt == 0) {                                 // (one barrier per thread, see osx7_kernel)
        os2::mbar_init(vbar, 1u);
        os2::mbar_init_fence();
    }
    const int c = gt & 15, h = gt >> 4;                                           // column of the strip, item index
    const int Nx = a.Nx, Nv = a.Nv, vmask = Nv - 1, np = a.np;
    const bool IP = IPM == 2 ? a.inplace != 0 : false;
    // (the FP32 pipe is what this kernel waits for most: the 15 twiddles of an item come from a 1.9 KB table in
    // shared memory, 15 loads per pass, instead of 11 complex products of four register-resident powers)
    for (int i = tid; i < 240; i += 768) twS[i] = __ldg(a.tw + i);               // (plan constants: before the wait)
    for (int k = tid; k < 129; k += 768) {
        const double2 cs = su.cs64[k];
        csS[k] = su.spline ? make_float4((float)cs.x, (float)cs.y, (float)(2.0 * cs.x * cs.x - 1.0), (float)(2.0 * cs.y * cs.x))
                           : make_float4((float)cs.x, (float)cs.y, (float)(2.0 - 2.0 * cs.x), 0.0f);
    }
    const float2* const twp = twS + h;            // [q-1][t], t = item index of passes A
    float2* const own = exch + h * W + c;                                     // position t = h
    constexpr int PS = 16 * W;                                                // float2 between positions 16 apart
    // Field solve fused into this kernel (su.fpart != NULL; grids of at most gridDim.x strips, one piece per CTA): the
    // exchange buffers of the three groups are free until the first pass A and hold, in this order, rho (Nx doubles),
    // the Green's function of the Fourier solve (Nx doubles, a plan constant: loaded before the wait) and the partial
    // sums of the convolution.
    // In-place mode (a.inplace: dst == src; vog_advect_v / vog_shift_v).  A strip's pairs are
    // stored in place as long as every window that still needs the overwritten rows is already on chip: the store of
    // pair p waits until the windows of pairs p - 1 and p + 1 have landed (landedS: last pair landed per group), and the
    // strip's first IPH rows, which the LAST pair's window reads again after the wrap, are kept in saveS.  That holds
    // for integer shifts up to IPB rows; a strip with larger shifts is written to the second grid a.dst2 instead and
    // flagged for the copy-back kernel (vog_os.cu strip_copy_kernel).
    // Pieces that are not whole strips (the balanced shares of the strips left over, or several CTAs per strip on narrow
    // grids) border on rows that ANOTHER CTA stores: a launch of osv7_halo_kernel in front of this one has copied the
    // IPH rows on either side of every such piece into a.halo (global scratch), and a piece's first / last window takes
    // the rows beyond its own range from there.  (A counter inside this kernel, on which every CTA arrives after saving
    // its own halos, did the same in one launch -- and deadlocks when two such grids share the GPU.)
    constexpr int IPH = os2::IPH, IPB = 24;
    __shared__ float saveS[IPH * W];
    __shared__ volatile int landedS[3];
    // the rows around a piece: lo = rows [Lw - IPH, Lw) below it, up = rows [Uw, Uw + IPH) behind it (original values;
    // whole strips: up = the strip's first rows in saveS); Lw = first row of the piece, Uw = first row behind it (unwrapped)
    struct Halo { const float* lo; const float* up; int Lw, Uw; };
    Halo hcur = {nullptr, saveS, 0, Nv};
    __shared__ float fusedE[W];
    __shared__ float4 srcRS[4 * W];               // delta-f source: (e^h, expm1 h, e^-h, expm1 -h), h = 16 rows, per (Gaussian, column)
    __shared__ float2 srcRV[4 * W];               // ... and (e^{g V}, expm1(g V)): block B from block A
    float* const fRho = reinterpret_cast<float*>(smem_raw + HEAD + RR * W * 4);
    float* const fGreen = reinterpret_cast<float*>(smem_raw + HEAD + GB + RR * W * 4);
    double* const fSum = reinterpret_cast<double*>(smem_raw + HEAD + 2 * GB + RR * W * 4);
    if (su.fpart)
        for (int i = tid; i < Nx; i += 768) fGreen[i] = (float)__ldg(su.green + i);
    if (tid < 5) asm volatile("prefetch.tensormap [%0];\n" ::"l"(reinterpret_cast<unsigned long long>(&maps.m[tid])) : "memory");

    const int G = gridDim.x, kb = blockIdx.x, nstrips = Nx / W;
    auto piece = [&](const int i, int& strip, int& q0, int& q1) -> bool {
        return osv7_piece(i, G, kb, nstrips, np, strip, q0, q1);
    };
    // S1 inside the kernel: the symbol table of a strip is COMPUTED here (no set-up kernel between the field solve and
    // this one).  Same arithmetic, entry for entry, as os_setup_v_kernel: beta, b, b* and the Everett / B-spline
    // coefficients in fp64 per column (32 threads: column x half; lane = the thread's index 0..31), then the 130
    // entries by fp32 Horner.  The fp64 part of piece i + 2 runs in ONE warp while piece i is being transformed.
    auto coeffs = [&](const int lane32, const int c0, float* const rec) {
        float* const afS = rec;
        int* const bS = reinterpret_cast<int*>(rec + 18 * W);
        float* const sS = rec + 19 * W;
        const int half = lane32 >> 4, cc = lane32 & 15, l = c0 + cc;
        double beta;
        float sshift = 0.0f;
        if (su.mode == 1) {
            double e = su.fpart ? (double)fusedE[cc] : (double)su.E[l];
            if (su.Eext) e += (double)su.Eext[l];
            beta = -e * su.dt / su.delta;
            sshift = (float)(su.dt * e);
        } else {
            beta = su.beta[l];
        }
        const double fl = floor(beta);
        const double tt0 = beta - fl;
        int bb;
        if (fabs(fl) < 9.0e18) {
            bb = (int)(__double2ll_rn(fl) & (long long)(su.N - 1));
        } else {
            double bm = fmod(fl, (double)su.N);
            if (bm < 0.0) bm += (double)su.N;
            bb = (int)bm;
            if (bb >= su.N) bb = 0;
        }
        if (half == 0) { bS[cc] = bb; sS[cc] = sshift; }
        if (!su.spline) {
            const double tt = half == 0 ? 1.0 - tt0 : tt0;
            double av = tt;
            constexpr double rcp[9] = {0.0, 1.0 / 6.0, 1.0 / 20.0, 1.0 / 42.0, 1.0 / 72.0, 1.0 / 110.0, 1.0 / 156.0,
                                       1.0 / 210.0, 1.0 / 272.0};            // 1 / (2m (2m+1))
            afS[(half * 9) * W + cc] = (float)av;
#pragma unroll
            for (int m = 1; m <= 8; ++m) {
                av = av * ((double)(m * m) - tt * tt) * rcp[m];
                afS[(half * 9 + m) * W + cc] = m <= su.d ? (float)av : 0.0f;
            }
        } else if (half == 0) {
            const double t = tt0, u = 1.0 - t;
            afS[0 * W + cc] = (float)(u * u * u / 6.0);
            afS[1 * W + cc] = (float)((4.0 - 6.0 * t * t + 3.0 * t * t * t) / 6.0);
            afS[2 * W + cc] = (float)((1.0 + 3.0 * t + 3.0 * t * t - 3.0 * t * t * t) / 6.0);
            afS[3 * W + cc] = (float)(t * t * t / 6.0);
        }
    };
    // where the raw rows of a piece lie: per-lane offset db, first row base (relative to pair start - HLO), row count
    struct Geo { int c0, base, nrows, db; bool gather; };
    auto geometry = [&](const int c0, const float* const rec) -> Geo {
        const int b = reinterpret_cast<const int*>(rec + 18 * W)[c];
        // spread of the shifts over the strip, as signed distances from column 0's (shifts live mod Nv)
        const int b0 = __shfl_sync(0xffffffffu, b, 0, 16);
        const int d = (((b - b0) + (Nv >> 1)) & vmask) - (Nv >> 1);
        int dmin = d, dmax = d;
#pragma unroll
        for (int o = 8; o > 0; o >>= 1) {
            dmin = min(dmin, __shfl_xor_sync(0xffffffffu, dmin, o));
            dmax = max(dmax, __shfl_xor_sync(0xffffffffu, dmax, o));
        }
        const int R = dmax - dmin;
        Geo g;
        g.c0 = c0;
        g.gather = R > RMAX;                       // uniform over the CTA (every half-warp sees the same 16 columns)
        // The union of the rows the 16 columns need is a box of the grid: 16 columns x (V + 256 + R) rows.  It is
        // requested by ONE thread of the group as a handful of 2-D tensor copies (cp.async.bulk.tensor, the TMA engine:
        // boxes of 256, 64, 16, 4 and 2 rows; a second run of boxes when the window wraps around the end of the
        // columns), counted in bytes on the group's mbarrier.  The per-thread 16-byte cp.async loop this replaces was
        // 18 % of all instructions the kernel executed (25 instructions of address arithmetic per copy).  A box must
        // start on a 128-byte boundary of shared memory = an even row of the raw buffer: the window starts on an even
        // row of the grid (one row early if need be) and holds an even number of rows.
        const int odd = g.gather ? 0 : ((b0 + dmin - HLO) & 1);
        g.db = g.gather ? 0 : d - dmin + odd;      // this lane's row offset inside the raw window
        g.base = g.gather ? b : b0 + dmin - odd;   // first raw row = pair start - HLO + base
        g.nrows = g.gather ? V + OS_LB : (V + OS_LB + R + odd + 1) & ~1;
        return g;
    };
    // request the raw rows of pair p: the union of the rows, unshifted (or, in the fallback, every lane its own rows)
    // mode (in place only): 1 = the rows below the piece come from hlo, 2 = the rows behind it from hup
    auto land = [&](const Geo& g, const int p, const int mode, const Halo& hl) {
        const float* const hlo = hl.lo;
        const float* const hup = hl.up;
        const int Lw = hl.Lw, Uw = hl.Uw;
        const int rs = p * (2 * V) - HLO + g.base;
        if (!g.gather) {
            // unwrapped first row of the window (the shift as a signed number), rows from the two halos
            const int urs = p * (2 * V) - HLO + (((g.base + (Nv >> 1)) & vmask) - (Nv >> 1));
            const int nA = (mode & 1) ? min(max(Lw - urs, 0), g.nrows) : 0;
            const int over = urs + g.nrows - Uw;
            const int nC = (mode & 2) ? min(max(over, 0), IPH) : 0;
            if (gt == 0) {
                os2::mbar_expect_tx(vbar, (unsigned)(g.nrows - nA - nC) * (W * 4u));
                // global rows: [urs + nA, e1) and, behind the upper halo, [Uw + nC, urs + nrows) (rows that only feed
                // discarded samples); each run wraps at the last row of the grid
                const int e1 = nC > 0 ? Uw : urs + g.nrows;
                for (int run = 0; run < 2; ++run) {
                    int ur = run == 0 ? urs + nA : Uw + nC;
                    const int ue = run == 0 ? e1 : urs + g.nrows;
                    if (run == 1 && nC == 0) break;
                    while (ur < ue) {
                        int gr = ur & vmask, sr = ur - urs;
                        int n = min(ue - ur, Nv - gr);               // (a window past the last row wraps to row 0)
                        ur += n;
#pragma unroll 1
                        for (int i = 0; i < 5; ++i) {
                            const int hb = os2::vbox_rows(i);
                            while (n >= hb) {
                                os2::tensor_g2s(raw + sr * W, &maps.m[i], g.c0, gr, vbar);
                                gr += hb; sr += hb; n -= hb;
                            }
                        }
                    }
                }
            }
            for (int i = gt; i < nA * W; i += 256) raw[i] = hlo[(IPH - nA) * W + i];
            for (int i = gt; i < nC * W; i += 256) raw[(Uw - urs) * W + i] = hup[i];
        } else {
            const float* const col = a.src + g.c0 + c;
            for (int r = h; r < g.nrows; r += 16) os2::cp_async4(raw + r * W + c, col + (size_t)((rs + r) & vmask) * Nx);
        }
    };

    OS_STAMP(0);
    OS_BLK(0);
    int strip, q0, q1, nstrip = 0, nq0 = 0, nq1 = 0;
    bool has = piece(0, strip, q0, q1), nhas = has && piece(1, nstrip, nq0, nq1);
    // Speculative first window.  The source grid is final before this CTA exists: this kernel's predecessor in the
    // stream (density or Poisson kernel) lets its dependents start only after its own wait on the kernel that wrote
    // the grid, so only E / rho need the wait below.  Each group requests, for its first pair, the rows that serve every
    // integer shift in [-SPEC, SPEC) -- the whole raw buffer -- while the field is still being solved; if the shifts
    // turn out larger (or spread too far) the window is requested again once they are known.
    constexpr int SPEC = (RR - OS_LB - V) / 2;     // 16 (Lagrange geometry) / 18 rows
    bool spec = false;
    if (su.spec && has && q0 + gid < q1) {
        Geo gs;
        gs.c0 = strip * W; gs.base = -SPEC; gs.nrows = RR; gs.db = 0; gs.gather = false;
        land(gs, q0 + gid, 0, hcur);
        spec = true;
    }
    pdl_wait();                                   // the field (or rho) comes from the kernel before
    pdl_launch_dependents();
    OS_STAMP(1);
    OS_BLK(1);
    int li_cur = 0;                                // pieces of this CTA that were not whole strips, so far
    if (su.fpart) {
        // S9 for the 16 columns of this strip.  rho_i (the density kernel's last blocks wrote it: dv * the slab sums in
        // the order of poisson_kernel) minus rho_0 (any constant only changes mode 0, which is dropped: P:205-211),
        // rounded to fp32 like poisson_kernel's input; E_i = sum_j G_{i-j} rho_j with G = the inverse transform of
        // 1 / (i k_m), modes 0 and Nx/2 dropped: the Fourier solve written as the circular convolution it is.
        // 48 shares of <= 43 products per column in fp32 (the fp64 pipe took 2.6 us for these 33 k multiply-adds), the
        // shares added in fp64 in a fixed order.
        const int xmask = Nx - 1, c0f = strip * W;
        const bool writer = has && q0 == 0;        // the strip's first segment publishes E and the energy share
        {
            const double ref = __ldcg(su.fpart);
            double r[3];                           // (Nx <= 16 gridDim.x <= 2368: three cells per thread, one round trip)
#pragma unroll
            for (int k = 0; k < 3; ++k) r[k] = tid + 768 * k < Nx ? __ldcg(su.fpart + tid + 768 * k) : 0.0;
#pragma unroll
            for (int k = 0; k < 3; ++k)
                if (tid + 768 * k < Nx) fRho[tid + 768 * k] = (float)(r[k] - ref);
            for (int i = tid + 2304; i < Nx; i += 768) fRho[i] = (float)(__ldcg(su.fpart + i) - ref);
            if (tid < 192) fRho[Nx + tid] = 0.0f;  // (the last chunks of the sum over j run past Nx)
        }
        __syncthreads();
        OS_STAMP(40);
        {
            // thread = (quad of columns cq, chunk of JC consecutive cells j): per cell one value of rho, one new value of G
            // (a rolling window of four) and four multiply-adds in fp32; the 8 chunks of a warp are folded by shuffles,
            // the 24 warps meet in shared memory; sums across threads in fp64, fixed order.
            const int cq = tid & 3, jp = tid >> 2, JC = (Nx + 191) / 192, j0 = jp * JC;
            const int gb = c0f + 4 * cq + 3 - j0;                      // index of G for column 4 cq + 3 at cell j0
            float g0 = fGreen[gb & xmask], g1 = fGreen[(gb - 1) & xmask], g2 = fGreen[(gb - 2) & xmask], g3;
            float a0 = 0.0f, a1 = 0.0f, a2 = 0.0f, a3 = 0.0f;        // columns 4 cq + 3, + 2, + 1, + 0
#pragma unroll 4
            for (int i = 0; i < JC; ++i) {
                g3 = fGreen[(gb - 3 - i) & xmask];
                const float rj = fRho[j0 + i];
                a0 = fmaf(g0, rj, a0); a1 = fmaf(g1, rj, a1); a2 = fmaf(g2, rj, a2); a3 = fmaf(g3, rj, a3);
                g0 = g1; g1 = g2; g2 = g3;
            }
            double d0 = (double)a0, d1 = (double)a1, d2 = (double)a2, d3 = (double)a3;
#pragma unroll
            for (int o = 16; o >= 4; o >>= 1) {
                d0 += __shfl_xor_sync(0xffffffffu, d0, o); d1 += __shfl_xor_sync(0xffffffffu, d1, o);
                d2 += __shfl_xor_sync(0xffffffffu, d2, o); d3 += __shfl_xor_sync(0xffffffffu, d3, o);
            }
            if ((tid & 28) == 0) {                 // lanes 0..3 of the warp: quad cq
                double* const o = fSum + (tid >> 5) * W + 4 * cq;
                o[3] = d0; o[2] = d1; o[1] = d2; o[0] = d3;
            }
        }
        __syncthreads();
        OS_STAMP(41);
        if (tid < 4 * W) {
            // 24 warp sums per column: four threads add six each, then the four meet by shuffles
            const int cc = tid >> 2, part = tid & 3;
            double sv = 0.0;
#pragma unroll
            for (int q = 0; q < 6; ++q) sv += fSum[(6 * part + q) * W + cc];
            sv += __shfl_xor_sync(0xffffffffu, sv, 1);
            sv += __shfl_xor_sync(0xffffffffu, sv, 2);
            if (part == 0) fusedE[cc] = (float)sv;
        }
        __syncthreads();
        if (tid < W) {
            const float ef = fusedE[tid];
            if (writer) {
                su.E_out[c0f + tid] = ef;
                if (su.energy_out) {   // (1/2) dx sum_i E_i^2: strip sums in strip order by the last strip to arrive
                    double e2 = (double)ef * (double)ef;
#pragma unroll
                    for (int o = 8; o > 0; o >>= 1) e2 += __shfl_xor_sync(0xffffu, e2, o);
                    if (tid == 0) {
                        su.e_part[strip] = e2;
                        __threadfence();
                        const unsigned n = atomicAdd(su.ticket, 1u);
                        if (n == (unsigned)nstrips - 1u) {
                            __threadfence();
                            double tot = 0.0;
                            for (int q = 0; q < nstrips; ++q) tot += __ldcg(su.e_part + q);
                            su.energy_out[0] = su.half_dx * tot;
                            *su.ticket = 0u;
                        }
                    }
                }
            }
        }
        __syncthreads();
    }
    OS_STAMP(2);
    if (tid < 2 * W && has) coeffs(tid, strip * W, cfS);
    if (tid >= 2 * W && tid < 4 * W && nhas) coeffs(tid - 2 * W, nstrip * W, cfS + CF);
    __syncthreads();
    OS_STAMP(3);
    bool pref = false;                             // the first window of this group in the current piece is on its way
    for (int it = 0; has; ++it) {
        const float* const rec = cfS + (it % 3) * CF;
        // the group's first window of the piece is requested first: it lands while the table is computed
        const Geo g = geometry(strip * W, rec);
        const float ssh = rec[19 * W + c];
        const int p0 = q0 + gid;
        bool ipok = false;
        const bool whole = q0 == 0 && q1 == np;
        if (IP) {
            const int sb = ((g.base + (Nv >> 1)) & vmask) - (Nv >> 1);     // first window row as a signed shift
            // (a piece's first window starts HLO - sb rows below the piece: at most the IPH rows of the lower halo)
            ipok = !g.gather && sb >= (whole ? -4 * IPB : HLO - IPH) && sb + (g.nrows - (V + OS_LB)) <= IPB;
            hcur.Lw = q0 * (2 * V);
            hcur.Uw = q1 < np ? q1 * (2 * V) : Nv;
            if (whole) {
                hcur.lo = nullptr;
                hcur.up = saveS;
            } else {
                hcur.lo = a.halo + (size_t)(kb * 4 + min(li_cur, 3)) * (2 * IPH * W);
                hcur.up = hcur.lo + IPH * W;
                ++li_cur;
            }
            if (tid < 3) landedS[tid] = -1;
            if (tid == 0 && !ipok) a.strip_flags[strip] = 1;
        }
        // which halos the window of pair p takes (in place): whole strips only the wrap behind the last row, and only for
        // windows requested after the strip's first stores; other pieces both sides, always
        auto lmode = [&](const int p) -> int {
            if (!IP || !ipok) return 0;
            if (whole) return p >= q0 + 3 ? 2 : 0;
            return (p == q0 ? 1 : 0) | (p == q1 - 1 ? 2 : 0);
        };
        int db_first = g.db;                       // row offset of this lane in the window of the group's first pair
        if (spec) {
            // does the speculative window hold the rows of every column?  first row needed by this lane, relative to
            // the window's first row: (base + db) - (-SPEC), base as a signed shift
            const int sb = (((g.base + (Nv >> 1)) & vmask) - (Nv >> 1)) + SPEC;
            const bool fits = !g.gather && sb >= 0 && sb + (g.nrows - (V + OS_LB)) <= RR - (V + OS_LB);
            if (fits) db_first = sb + g.db;
            else {                                 // (uniform over the CTA: every half-warp sees the same 16 columns)
                os2::mbar_wait(vbar, vpar); vpar ^= 1u;
                os2::bar_group(gid + 1);           // (nobody of the group may still be waiting when the barrier is re-armed)
                land(g, p0, 0, hcur);
            }
            spec = false;
        } else if (!pref && p0 < q1) land(g, p0, lmode(p0), hcur);
        pref = false;
        if (IP && whole)                           // (behind the first requests: the table barrier below orders it before any store)
            for (int i = tid; i < IPH * W; i += 768)
                saveS[i] = __ldcg(a.src + (size_t)(i >> 4) * Nx + g.c0 + (i & (W - 1)));
        if (tid >= 768 - 6 * a.ng * W) {
            // delta-f source constants of (Gaussian gg, column cc): same expressions as osv2_source without a table,
            // one transcendental per thread (two warps computing all six per entry were the slowest of this phase), in
            // the CTA's last threads, which have two table entries below instead of three
            const int ti = tid - (768 - 6 * a.ng * W);
            const int which = ti / (a.ng * W), i = ti - which * (a.ng * W), cc = i & (W - 1), gg = i >> 4;
            const float cgs = a.cg4[gg] * rec[19 * W + cc];
            const float hh = 32.0f * cgs * a.dvf, hv = 2.0f * (float)V * cgs * a.dvf;
            const float arg = which < 2 ? hh : (which < 4 ? -hh : hv);
            const float val = (which & 1) ? expm1f(arg) : expf(arg);
            if (which < 4) reinterpret_cast<float*>(srcRS)[4 * i + which] = val;
            else reinterpret_cast<float*>(srcRV)[2 * i + (which - 4)] = val;
        }
        // ---- the strip's table: 130 x 16 entries.  A thread's entries all belong to column tid & 15 (768 is a multiple
        // of 16): its 18 coefficients are read once.
        {
            const int cc = tid & 15;
            float cfr[18];
#pragma unroll
            for (int j = 0; j < 18; ++j) cfr[j] = rec[j * W + cc];
#pragma unroll 1
            for (int kk = tid >> 4; kk < OS_LAMW; kk += 48) {
                float2 o;
                if (kk == 129) o = make_float2(rec[18 * W + cc], rec[19 * W + cc]);
                else if (kk == 0) o = make_float2(1.0f / (float)OS_LB, 0.0f);          // lambda_0 = sum of the weights = 1
                else {
                    const float4 cs = csS[kk];
                    const float cf = cs.x, sn = cs.y;
                    float lr, li;
                    if (su.spline) {
                        const float Bm1 = cfr[0], B0 = cfr[1], B1 = cfr[2], B2 = cfr[3];
                        const float gg = 3.0f / (2.0f + cf);
                        lr = fmaf(B2, cs.z, fmaf(Bm1 + B1, cf, B0)) * gg;
                        li = fmaf(B2, cs.w, (B1 - Bm1) * sn) * gg;
                    } else {
                        const float sv = cs.z;
                        float h0 = 0.0f, h1 = 0.0f;
#pragma unroll
                        for (int j = 8; j >= 0; --j) {
                            h0 = fmaf(h0, sv, cfr[j]);
                            h1 = fmaf(h1, sv, cfr[9 + j]);
                        }
                        lr = fmaf(cf, h1, h0);
                        li = sn * h1;
                    }
                    o = make_float2(lr * (1.0f / (float)OS_LB), li * (1.0f / (float)OS_LB));
                }
                lamS[kk * W + cc] = o;
            }
        }
        OS_STAMP(42);
        __syncthreads();                           // table visible to everybody
        OS_STAMP(4);
        if (it == 0) OS_BLK(2);
        // the piece after next: its fp64 coefficients, in the last warp, while everybody else transforms
        int fstrip = 0, fq0 = 0, fq1 = 0;
        const bool fhas = nhas && piece(it + 2, fstrip, fq0, fq1);
        if (tid >= 768 - 2 * W && fhas) coeffs(tid - (768 - 2 * W), fstrip * W, cfS + ((it + 2) % 3) * CF);
        Geo gn = g;
        if (nhas) gn = geometry(nstrip * W, cfS + ((it + 1) % 3) * CF);
        const int np0 = nq0 + gid;
        float* const ocol = ((IP && !ipok) ? a.dst2 : a.dst) + g.c0 + c;
        for (int p = p0; p < q1; p += 3) {
            if (g.gather) os2::cp_async_wait_all();
            else { os2::mbar_wait(vbar, vpar); vpar ^= 1u; }
            if (IP && ipok && gt == 0) landedS[gid] = p;
            OS_STAMP(5 + 4 * ((p - p0) / 3));
            os2::bar_group(gid + 1);               // raw rows of pair p visible; exchange buffer of the last pair read
            // ---- pass A (item t = h): samples from the raw rows with this lane's offset
            {
                float2 x[16];
                const float* const rp = raw + (h + db_first) * W + c;
                db_first = g.db;
#pragma unroll
                for (int k = 0; k < 16; ++k) x[k] = make_float2(rp[16 * k * W], rp[(16 * k + V) * W]);
                dft_dif<16, 1>(x);
                own[0] = x[0];
#pragma unroll
                for (int q = 1; q < 16; ++q) own[q * PS] = cmul(x[brev(q, 16)], twp[(q - 1) * 16]);
            }
            os2::bar_group(gid + 1);               // exchange buffer complete; raw rows all read
            OS_STAMP(6 + 4 * ((p - p0) / 3));
            // the next window lands behind the middle stage and the inverse pass: this piece's, or -- after the group's
            // last pair of the piece -- the group's first of the NEXT piece (its shifts are known two pieces ahead)
            if (p + 3 < q1) land(g, p + 3, lmode(p + 3), hcur);
            else if (nhas && np0 < nq1) {
                // the group's first window of the NEXT piece.  In place, a piece that is not a whole strip takes the rows
                // beyond its range from its halo slot (saved before this kernel started), if its shifts allow in-place
                // storing at all -- the same test as at the top of the piece, on the next piece's geometry.
                int nmode = 0;
                Halo hn = hcur;
                if (IP && !(nq0 == 0 && nq1 == np)) {
                    const int sbn = ((gn.base + (Nv >> 1)) & vmask) - (Nv >> 1);
                    const bool okn = !gn.gather && sbn >= HLO - IPH && sbn + (gn.nrows - (V + OS_LB)) <= IPB;
                    hn.lo = a.halo + (size_t)(kb * 4 + min(li_cur, 3)) * (2 * IPH * W);
                    hn.up = hn.lo + IPH * W;
                    hn.Lw = nq0 * (2 * V);
                    hn.Uw = nq1 < np ? nq1 * (2 * V) : Nv;
                    if (okn) nmode = (np0 == nq0 ? 1 : 0) | (np0 == nq1 - 1 ? 2 : 0);
                }
                land(gn, np0, nmode, hn);
                pref = true;
            }
            // ---- middle stage (item g = h): positions 16 g + j
            {
                float2* const sp = exch + h * 16 * W + c;
                float2 x[16];
#pragma unroll
                for (int j = 0; j < 16; ++j) x[j] = sp[j * W];
                os2::mid16<W>(x, lamS + c, h);
#pragma unroll
                for (int j = 0; j < 16; ++j) sp[j * W] = x[j];
            }
            if (IP && ipok && gt == 0) {           // in place: the neighbours' windows must be on chip before these rows change
                // (publishing a group's window in flight as soon as its barrier completes, instead of when the group
                // gets to it, was measured: 144 -> 149 us at 8192^2, the polling costs more than the wait)
                if (p + 1 < q1) while (landedS[(gid + 1) % 3] < p + 1) { }
                if (p > q0) while (landedS[(gid + 2) % 3] < p - 1) { }
            }
            os2::bar_group(gid + 1);
            OS_STAMP(7 + 4 * ((p - p0) / 3));
            // ---- inverse pass A (item j = h): kept samples -> rows of the destination
            {
                float2 x[16];
                x[0] = own[0];
#pragma unroll
                for (int q = 1; q < 16; ++q) x[brev(q, 16)] = cmulc(own[q * PS], twp[(q - 1) * 16]);
                idft_dit<16, 1>(x);
                const int r0 = p * (2 * V) + h - HLO;          // row of sample n = t = h of block A
                if (a.ng > 0) osv2_source<V, HLO, W>(x, a, srcRS, c, r0, ssh, srcRV);
                float* const po = ocol + (ptrdiff_t)r0 * Nx;
                if ((p + 1) * (2 * V) <= Nv) os2_store_v_full<V, HLO>(po, (size_t)Nx, h, x);
                else os2_store_v<V, HLO>(po, (size_t)Nx, r0, Nv, h, false, x);
            }
            OS_STAMP(8 + 4 * ((p - p0) / 3));
        }
        __syncthreads();                           // every group is done with the table of this piece
        OS_STAMP(30);
        OS_BLK(3);
        has = nhas; strip = nstrip; q0 = nq0; q1 = nq1;
        nhas = fhas; nstrip = fstrip; nq0 = fq0; nq1 = fq1;
    }
}

}  // namespace vog
