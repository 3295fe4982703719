// vog_os.cuh -- overlap-save advection kernels (line length N >= 1024).
// Product code; shares nothing with oracle/.
//
// The circulant interpolation matrix A of P:98-100 has a SHORT first row: 2d+2 non-zeros for Lagrange
// 2d+1, and an exponentially decaying one for the cubic spline (|a_j| ~ 0.268^|j|,
// P:117-129).  u' = A u is therefore a short cyclic convolution, and the Fourier-space product of
// P:131-149 can be taken block-wise (overlap-save): every block of LB = 256 samples of the rolled line
// r_i = u_{i+b} is transformed, multiplied by the symbol lambda(theta_k), theta_k = 2 pi k / LB, and
// transformed back; the V = 224 samples in the middle of the block are exactly (Lagrange) or to
// <= 2e-9 max|u| (spline: the neglected tail of the row, far below fp32 rounding) the samples
// of A u, the H = 16 on either side are discarded.  Compared with one length-N transform per line:
//   * 8 instead of log2(N) butterfly levels, two passes instead of three, no big twiddle table;
//   * the symbol is a per-line table lam[k], k = 0..128, written by the setup kernel (shift split and
//     interpolation coefficients in fp64, the 129 entries in fp32) and shared by all blocks of the line --
//     no polynomial evaluation in the hot loop;
//   * the integer part b of the shift is folded into the load address ("integer roll by
//     index"): no rotation factor at all (x keeps a residual br in {-2..1} in the table to stay 128-bit aligned);
//   * the working set of a block is 1 KB per line, so the strided (v) direction can use strips 32 columns
//     wide at ANY Nv: full 128-byte lines, no shared-memory capacity limit.
// x-direction: even/odd packing (a block is 128 complex), CTA owns whole lines, in place.
// v-direction: 32 adjacent columns = the 32 lanes of a warp, the same even/odd block transform per column;
//   OUT of place (src != dst): a block reads rows that other blocks write, so in-place would race.
// Both kernels land their input asynchronously (cp.async) in the scratch slots that the landing thread
// itself transforms, and start landing the next work unit as soon as those slots have been read back.
#pragma once
#include "vog_fft.cuh"
#include "vog_internal.h"

namespace vog {

__device__ __forceinline__ void os_cp_async16(void* smem, const void* gmem)
{
    const unsigned s = (unsigned)__cvta_generic_to_shared(smem);
    asm volatile("cp.async.ca.shared.global [%0], [%1], 16;\n" ::"r"(s), "l"(gmem) : "memory");
}
__device__ __forceinline__ void os_cp_async16_cg(void* smem, const void* gmem)
{
    const unsigned s = (unsigned)__cvta_generic_to_shared(smem);
    asm volatile("cp.async.cg.shared.global [%0], [%1], 16;\n" ::"r"(s), "l"(gmem) : "memory");
}
__device__ __forceinline__ void os_cp_async_commit_wait()
{
    asm volatile("cp.async.commit_group;\ncp.async.wait_group 0;\n" ::: "memory");
}

// One mirror pair (k, M-k) of the half-length spectrum of an even/odd packed real block:
// untangle, multiply by the tabulated symbol, re-tangle.  P = Z_k, Qm = Z_{M-k}; cs = (cos, sin)(2 pi k/LB);
// a = lambda_k/(2 LB), cc = conj(lambda_{M-k})/(2 LB).
__device__ __forceinline__ void os_pair_x(float2& P, float2& Qm, const float2 cs, const float2 a, const float2 cc)
{
    const float2 Qc = make_float2(Qm.x, -Qm.y);                     // conj(Z_{M-k})
    const float2 E2 = cadd(P, Qc), D2 = csub(P, Qc);
    // T2 = W_N^k (-i D2), W_N^k = (c, -s):  (-i D2) conj((c, s))
    const float2 T2 = cmulc(make_float2(D2.y, -D2.x), cs);
    const float2 Up = cadd(E2, T2), Um = csub(E2, T2);
    const float2 Vp = cmul(Up, a), Vm = cmul(Um, cc);
    const float2 Ep = cadd(Vp, Vm), Dp = csub(Vp, Vm);
    const float2 Op = cmul(Dp, cs);                                 // conj(W) Dp
    P = cadd(Ep, make_float2(-Op.y, Op.x));                         // E' + i O'
    const float2 R = csub(Ep, make_float2(-Op.y, Op.x));            // E' - i O'
    Qm = make_float2(R.x, -R.y);
}


// ---------------------------------------------------------------------------------------------
// x-direction.  Block of LB = 256 reals = 128 complex = radix 8 (stride 16) x radix 16.
// Scratch: 64 chunks (1 KB) per block; logical chunk = group*8 + j (group = radix-8 output index,
// j = pair of positions inside the group); physical chunk = group*8 + (j ^ key(block, group)).
// key: groups 0 and 4 (the "special" middle-stage item of a block): block & 7; groups g and 8-g,
// g = 1..3 (item u = g): (3 block + g - 1) & 7.  With the item orders used below, the 8 lanes of every
// quarter-warp hit 8 distinct 16-byte bank groups in all three phases.
namespace osx {
constexpr int MB = OS_LB / 2;      // complex length of a block
constexpr int CPB = MB / 2;        // chunks per block (64)
constexpr int VC = OS_V / 4;       // valid chunks per block (56)
constexpr int HC = OS_H / 4;       // halo chunks (4)
}

// slots of one pass-A item: sl[c] = (block base + (tp ^ key_c)), c = 0: groups 0,4; c = 1..3: groups c, 8-c
struct OsxSlots { int s[4]; };
__device__ __forceinline__ OsxSlots osx_slots(const int lb, const int tp)
{
    OsxSlots r;
    const int cb = lb * osx::CPB, k3 = 3 * lb;
    r.s[0] = cb + (tp ^ (lb & 7));
    r.s[1] = cb + (tp ^ (k3 & 7));
    r.s[2] = cb + (tp ^ ((k3 + 1) & 7));
    r.s[3] = cb + (tp ^ ((k3 + 2) & 7));
    return r;
}
__host__ __device__ constexpr int osx_cls(int g) { return (g & 3) == 0 ? 0 : (g < 4 ? g : 8 - g); }

// asynchronous landing of one item's 8 window chunks in the scratch slots the SAME thread transforms in
// pass A and reads again in the inverse pass (window chunk tp + 8k <-> slot of (group k, tp)): no other
// thread touches these slots between the inverse pass of one line group and pass A of the next.
__device__ __forceinline__ void osx_land(float4* __restrict__ scr, const OsxSlots sl, const float4* __restrict__ gline,
                                         const int mask, const int wc)
{
#pragma unroll
    for (int k = 0; k < 8; ++k)
        os_cp_async16_cg(scr + sl.s[osx_cls(k)] + k * 8, gline + ((wc + 8 * k) & mask));
}

// forward pass A of one item: two adjacent radix-8 butterflies (positions 2tp, 2tp+1 + 16k), in place
__device__ __forceinline__ void osx_fwd(float4* __restrict__ scr, const OsxSlots sl,
                                        const int tp, const float2* __restrict__ twS)
{
    float2 x0[8], x1[8];
#pragma unroll
    for (int k = 0; k < 8; ++k) {
        const float4 v = scr[sl.s[osx_cls(k)] + k * 8];
        x0[k] = make_float2(v.x, v.y);
        x1[k] = make_float2(v.z, v.w);
    }
    dft_dif<8, 1>(x0);
    dft_dif<8, 1>(x1);
    scr[sl.s[0]] = make_float4(x0[0].x, x0[0].y, x1[0].x, x1[0].y);
    const float4* __restrict__ tw4 = reinterpret_cast<const float4*>(twS) + tp;
#pragma unroll
    for (int q = 1; q < 8; ++q) {
        const float4 w = tw4[(q - 1) * 8];
        const float2 y0 = cmul(x0[brev(q, 8)], make_float2(w.x, w.y));
        const float2 y1 = cmul(x1[brev(q, 8)], make_float2(w.z, w.w));
        scr[sl.s[osx_cls(q)] + q * 8] = make_float4(y0.x, y0.y, y1.x, y1.y);
    }
}

// inverse pass A of one item; stores the valid chunks of the block (+ the block mean dc)
__device__ __forceinline__ void osx_inv(float4* __restrict__ gline, const int nchunk, const int oc0,
                                        const float4* __restrict__ scr, const OsxSlots sl, const int tp,
                                        const float2* __restrict__ twS, const float dc)
{
    float2 x0[8], x1[8];
    {
        const float4 v = scr[sl.s[0]];
        x0[0] = make_float2(v.x, v.y);
        x1[0] = make_float2(v.z, v.w);
    }
    const float4* __restrict__ tw4 = reinterpret_cast<const float4*>(twS) + tp;
#pragma unroll
    for (int q = 1; q < 8; ++q) {
        const float4 v = scr[sl.s[osx_cls(q)] + q * 8];
        const float4 w = tw4[(q - 1) * 8];
        x0[brev(q, 8)] = cmulc(make_float2(v.x, v.y), make_float2(w.x, w.y));
        x1[brev(q, 8)] = cmulc(make_float2(v.z, v.w), make_float2(w.z, w.w));
    }
    idft_dit<8, 1>(x0);
    idft_dit<8, 1>(x1);
    const float2 d2 = make_float2(dc, dc);
#pragma unroll
    for (int k = 0; k < 8; ++k) {
        const int c = tp + 8 * k;                    // chunk inside the window
        const int oc = oc0 + c - osx::HC;            // chunk of the line
        if (c >= osx::HC && c < osx::HC + osx::VC && oc < nchunk) {
            const float2 a = cadd(x0[k], d2), b = cadd(x1[k], d2);
            __stcs(gline + oc, make_float4(a.x, a.y, b.x, b.y));
        }
    }
}
// middle stage of one item (two mirror groups gA, gB of 16 complex): radix 16, untangle, symbol,
// re-tangle, inverse radix 16.  XA[brev q] = Z_{kA + 8 q}, XB[brev q] = Z_{kB + 8 q}.
//   normal item u = 1..3: gA = u, gB = 8 - u; pairs (XA[brev q], XB[brev(15-q)]), k = u + 8 q.
//   SPECIAL item: gA = 0, gB = 4 (its own mirror): pairs (XB[brev q], XB[brev(15-q)]), k = 4 + 8 q, q < 8;
//     (XA[brev q], XA[brev(16-q)]), k = 8 q, q = 1..7; k = 64 mirrors itself; k = 0 (with k = 128) apart.
template <bool SPECIAL>
__device__ __forceinline__ void osx_mid(float4* __restrict__ scr, const int cb, const int key, const int u,
                                        const float2* __restrict__ lamS, const float2* __restrict__ csS,
                                        float* __restrict__ dc)
{
    constexpr int M = osx::MB, ML = M / 16;          // 128, 8
    const int gA = SPECIAL ? 0 : u, gB = SPECIAL ? 4 : 8 - u;
    float4* const pa = scr + cb + gA * 8;
    float4* const pb = scr + cb + gB * 8;
    float2 XA[16], XB[16];
#pragma unroll
    for (int j = 0; j < 8; ++j) {
        const float4 va = pa[j ^ key], vb = pb[j ^ key];
        XA[2 * j] = make_float2(va.x, va.y); XA[2 * j + 1] = make_float2(va.z, va.w);
        XB[2 * j] = make_float2(vb.x, vb.y); XB[2 * j + 1] = make_float2(vb.z, vb.w);
    }
    dft_dif<16, 1>(XA);
    dft_dif<16, 1>(XB);
    if constexpr (!SPECIAL) {
#pragma unroll
        for (int q = 0; q < 16; ++q) {
            const int k = u + ML * q;
            const float2 lm = lamS[M - k];
            os_pair_x(XA[brev(q, 16)], XB[brev(15 - q, 16)], csS[k], lamS[k], make_float2(lm.x, -lm.y));
        }
    } else {
#pragma unroll
        for (int q = 0; q < 8; ++q) {
            const int k = ML / 2 + ML * q;
            const float2 lm = lamS[M - k];
            os_pair_x(XB[brev(q, 16)], XB[brev(15 - q, 16)], csS[k], lamS[k], make_float2(lm.x, -lm.y));
        }
#pragma unroll
        for (int q = 1; q < 8; ++q) {
            const int k = ML * q;
            const float2 lm = lamS[M - k];
            os_pair_x(XA[brev(q, 16)], XA[brev(16 - q, 16)], csS[k], lamS[k], make_float2(lm.x, -lm.y));
        }
        {
            const float2 lm = lamS[M / 2];
            float2 dup = XA[brev(8, 16)];
            os_pair_x(XA[brev(8, 16)], dup, csS[M / 2], lm, make_float2(lm.x, -lm.y));
        }
        // block modes 0 and LB/2: U_0 = x + y, U_M = x - y; lambda_0 = 1 exactly (lam[0] = (1/(2 LB), 0)).
        // The block mean A0 by-passes the inverse transform and is added back in the last pass.
        const float2 z0 = XA[0];
        const float A0 = 2.0f * lamS[0].x * (z0.x + z0.y), Bn = 2.0f * lamS[M].x * (z0.x - z0.y);
        XA[0] = make_float2(Bn, -Bn);
        *dc = A0;
    }
    idft_dit<16, 1>(XA);
    idft_dit<16, 1>(XB);
#pragma unroll
    for (int j = 0; j < 8; ++j) {
        pa[j ^ key] = make_float4(XA[2 * j].x, XA[2 * j].y, XA[2 * j + 1].x, XA[2 * j + 1].y);
        pb[j ^ key] = make_float4(XB[2 * j].x, XB[2 * j].y, XB[2 * j + 1].x, XB[2 * j + 1].y);
    }
}

// Persistent kernel: one iteration = lpi whole lines (a CTA owns whole lines, so src may equal dst: all
// loads of a line happen before the barrier that precedes its first store).
__global__ void __launch_bounds__(128, 4) osx_kernel(const OsArgs a)
{
    extern __shared__ __align__(16) unsigned char smem_raw[];
    const int lpi = a.lpi, nb = a.nb, nblk = lpi * nb;
    float4* const scr = reinterpret_cast<float4*>(smem_raw);                        // nblk*64 chunks
    float2* const lamS = reinterpret_cast<float2*>(scr + nblk * osx::CPB);          // lpi*OS_LAMW
    float2* const csS = lamS + lpi * OS_LAMW;                                       // 130
    float2* const twS = csS + 130;                                                  // 7*16
    float* const dcS = reinterpret_cast<float*>(twS + 112);                         // nblk
    const int tid = threadIdx.x, T = blockDim.x;
    const int nchunk = a.N >> 2;
    const unsigned inv_nb = a.inv_nb;      // ceil(2^16 / nb): lb / nb == (lb * inv_nb) >> 16 for lb < 2^12

    for (int i = tid; i < 129; i += T) csS[i] = __ldg(a.cs + i);
    for (int i = tid; i < 112; i += T) twS[i] = __ldg(a.tw + i);

    const int nA = nblk * 8;
    // window chunk of item w of the line group starting at line0, and the landing of all of a thread's items
    auto land = [&](const int w, const int line0) {
        const int lb = w >> 3, tp = w & 7;
        const int l = (int)(((unsigned)lb * inv_nb) >> 16), blk = lb - l * nb;
        const int b4 = __float_as_int(__ldg(&a.lam[(size_t)(line0 + l) * OS_LAMW + 129].x));
        const float4* gline = reinterpret_cast<const float4*>(a.src) + (size_t)(line0 + l) * nchunk;
        osx_land(scr, osx_slots(lb, tp), gline, nchunk - 1, osx::VC * blk - osx::HC + b4 + tp);
    };
    if ((int)blockIdx.x < a.n_groups)
        for (int w = tid; w < nA; w += T) land(w, blockIdx.x * lpi);
    __syncthreads();                               // csS, twS visible
    for (int g = blockIdx.x; g < a.n_groups; g += gridDim.x) {
        const int line0 = g * lpi;
        // (the symbol tables and dcS of the previous group were last read before / are rewritten after a
        // barrier of this iteration, so no barrier is needed here)
        {
            const float4* src4 = reinterpret_cast<const float4*>(a.lam + (size_t)line0 * OS_LAMW);
            float4* dst4 = reinterpret_cast<float4*>(lamS);
            for (int i = tid; i < lpi * (OS_LAMW / 2); i += T) os_cp_async16(dst4 + i, src4 + i);
        }
        os_cp_async_commit_wait();                 // this thread's window chunks (and table rows) have landed
        // ---- pass A: scratch -> registers -> scratch, every thread on the slots it landed itself
#pragma unroll 1
        for (int w = tid; w < nA; w += T) osx_fwd(scr, osx_slots(w >> 3, w & 7), w & 7, twS);
        __syncthreads();
        // ---- middle stage: items [0, nblk) are the special items of the blocks, then 3 per block
#pragma unroll 1
        for (int w = tid; w < nblk * 4; w += T) {
            if (w < nblk) {
                const int l = (int)(((unsigned)w * inv_nb) >> 16);
                osx_mid<true>(scr, w * osx::CPB, w & 7, 0, lamS + l * OS_LAMW, csS, dcS + w);
            } else {
                const int wp = w - nblk;
                const int lb = (int)(((unsigned)wp * 43691u) >> 17), u = wp - 3 * lb + 1;   // wp / 3 (wp < 2^15)
                const int l = (int)(((unsigned)lb * inv_nb) >> 16);
                osx_mid<false>(scr, lb * osx::CPB, wp & 7, u, lamS + l * OS_LAMW, csS, nullptr);
            }
        }
        __syncthreads();
        // ---- inverse pass A: scratch -> registers -> global; as soon as an item's slots are read, the
        // same item of the NEXT line group starts landing in them (hidden behind the rest of this pass).
        // In place this is safe: every load of THIS group completed before the barrier after pass A, and
        // the next group is other lines.
        const int gn = g + gridDim.x;
#pragma unroll 1
        for (int w = tid; w < nA; w += T) {
            const int lb = w >> 3, tp = w & 7;
            const int l = (int)(((unsigned)lb * inv_nb) >> 16), blk = lb - l * nb;
            float4* gline = reinterpret_cast<float4*>(a.dst) + (size_t)(line0 + l) * nchunk;
            osx_inv(gline, nchunk, osx::VC * blk, scr, osx_slots(lb, tp), tp, twS, dcS[lb]);
            if (gn < a.n_groups) land(w, gn * lpi);
        }
    }
}

// ---------------------------------------------------------------------------------------------
// v-direction.  A strip is 32 adjacent columns = the 32 lanes of a warp; every lane advects ITS column with
// even/odd packing along v (z_n = f[2n][c] + i f[2n+1][c], the same 128-complex block transform as in x).
//   * a row of the strip is one 128-byte line: every global load and store is fully coalesced, and a
//     lane applies its own integer shift b_c by addressing (rows r + b_c);
//   * scratch is [position][lane] float2: all shared accesses are conflict-free without padding;
//   * an item type (radix-8 butterfly t, middle-stage item u) is uniform across a warp: no divergence
//     between the "special" and the normal middle-stage items;
//   * the symbol tables arrive transposed ([k][column], written that way by the setup kernel).
// Out of place (src != dst): a block reads rows that other blocks write.
namespace osv {
constexpr int MB = OS_LB / 2;          // complex per block and column (128)
constexpr int W = 32;                  // columns per strip
constexpr int HN = OS_H / 2;           // halo in complex samples (8)
constexpr int VN = OS_V / 2;           // valid complex samples per block (112)
}

template <bool SPECIAL>
__device__ __forceinline__ void osv_mid(float2* __restrict__ scr, const int u, const float2* __restrict__ lamS,
                                        const float2* __restrict__ csS, float* __restrict__ dc)
{
    constexpr int M = osv::MB, ML = M / 16, W = osv::W;     // 128, 8
    const int gA = SPECIAL ? 0 : u, gB = SPECIAL ? 4 : 8 - u;
    float2* const pa = scr + gA * 16 * W;
    float2* const pb = scr + gB * 16 * W;
    float2 XA[16], XB[16];
#pragma unroll
    for (int j = 0; j < 16; ++j) { XA[j] = pa[j * W]; XB[j] = pb[j * W]; }
    dft_dif<16, 1>(XA);
    dft_dif<16, 1>(XB);
    if constexpr (!SPECIAL) {
#pragma unroll
        for (int q = 0; q < 16; ++q) {
            const int k = u + ML * q;
            const float2 lm = lamS[(M - k) * W];
            os_pair_x(XA[brev(q, 16)], XB[brev(15 - q, 16)], csS[k], lamS[k * W], make_float2(lm.x, -lm.y));
        }
    } else {
#pragma unroll
        for (int q = 0; q < 8; ++q) {
            constexpr int k0 = ML / 2;
            const int k = k0 + ML * q;
            const float2 lm = lamS[(M - k) * W];
            os_pair_x(XB[brev(q, 16)], XB[brev(15 - q, 16)], csS[k], lamS[k * W], make_float2(lm.x, -lm.y));
        }
#pragma unroll
        for (int q = 1; q < 8; ++q) {
            const int k = ML * q;
            const float2 lm = lamS[(M - k) * W];
            os_pair_x(XA[brev(q, 16)], XA[brev(16 - q, 16)], csS[k], lamS[k * W], make_float2(lm.x, -lm.y));
        }
        {
            const float2 lm = lamS[(M / 2) * W];
            float2 dup = XA[brev(8, 16)];
            os_pair_x(XA[brev(8, 16)], dup, csS[M / 2], lm, make_float2(lm.x, -lm.y));
        }
        const float2 z0 = XA[0];
        const float A0 = 2.0f * lamS[0].x * (z0.x + z0.y), Bn = 2.0f * lamS[M * W].x * (z0.x - z0.y);
        XA[0] = make_float2(Bn, -Bn);
        *dc = A0;                                   // block mean of this column, added back in the last pass
    }
    idft_dit<16, 1>(XA);
    idft_dit<16, 1>(XB);
#pragma unroll
    for (int j = 0; j < 16; ++j) { pa[j * W] = XA[j]; pb[j * W] = XB[j]; }
}

__device__ __forceinline__ void os_cp_async4(void* smem, const void* gmem)
{
    const unsigned s = (unsigned)__cvta_generic_to_shared(smem);
    asm volatile("cp.async.ca.shared.global [%0], [%1], 4;\n" ::"r"(s), "l"(gmem) : "memory");
}

// asynchronous landing of one item (butterfly t of a block, this lane's column): sample n = t + 16 k is rows
// r0 + 32 k and r0 + 32 k + 1 of the column.  It lands in the 256 bytes of position n that this WARP (32
// columns, same t) transforms in pass A and reads again in the inverse pass -- planar (32 real parts, then 32
// imaginary parts) so that the 4-byte copies of a warp are bank-conflict free; pass A reads the planar
// words and writes the position back as interleaved float2 (all reads of a warp precede its writes).
__device__ __forceinline__ void osv_land(float* __restrict__ pw, const float* __restrict__ col, const int Nx,
                                         const int vmask, const int r0)
{
    constexpr int W = osv::W;
    const int rr = r0 & vmask;
    if (rr + OS_LB <= vmask) {                      // the window does not wrap: constant row stride
        const float* p = col + rr * Nx;
        const int s32 = 32 * Nx;
#pragma unroll
        for (int k = 0; k < 8; ++k) {
            os_cp_async4(pw + k * 16 * W * 2, p);
            os_cp_async4(pw + k * 16 * W * 2 + W, p + Nx);
            p += s32;
        }
    } else {
#pragma unroll
        for (int k = 0; k < 8; ++k) {
            const int ra = (r0 + 32 * k) & vmask, rb = (r0 + 32 * k + 1) & vmask;
            os_cp_async4(pw + k * 16 * W * 2, col + ra * Nx);
            os_cp_async4(pw + k * 16 * W * 2 + W, col + rb * Nx);
        }
    }
}

// pw = planar words of position t for this lane (float index (pos * 32) * 2 + lane); o = the same position as
// interleaved float2 for this lane
__device__ __forceinline__ void osv_fwd(const float* __restrict__ pw, float2* __restrict__ o,
                                        const float2* __restrict__ tw)
{
    constexpr int W = osv::W;
    float2 x[8];
#pragma unroll
    for (int k = 0; k < 8; ++k) x[k] = make_float2(pw[k * 16 * W * 2], pw[k * 16 * W * 2 + W]);
    dft_dif<8, 1>(x);
    o[0] = x[0];
#pragma unroll
    for (int q = 1; q < 8; ++q) o[q * 16 * W] = cmul(x[brev(q, 8)], tw[(q - 1) * 16]);
}

// T = 128 rb threads: warp w handles butterflies t = w, w + nw, .. of the rb blocks of a group
__global__ void __launch_bounds__(256, 2) osv_kernel(const OsArgs a)
{
    extern __shared__ __align__(16) unsigned char smem_raw[];
    constexpr int W = osv::W, MB = osv::MB;
    const int rb = a.rb, nb = a.nb;
    float2* const scr = reinterpret_cast<float2*>(smem_raw);                  // rb * 128 * 32
    float2* const lamS = scr + rb * MB * W;                                   // 130 * 32, [k][lane]
    float2* const csS = lamS + OS_LAMW * W;                                   // 130
    float2* const twS = csS + 130;                                            // 7 * 16
    float* const dcS = reinterpret_cast<float*>(twS + 112);                   // rb * 32
    const int tid = threadIdx.x, T = blockDim.x, lane = tid & 31, wid = tid >> 5, nw = T >> 5;
    const int Nx = a.Nx, Nv = a.Nv, vmask = Nv - 1;
    const int c0 = blockIdx.x * W;

    {   // symbol tables of the 32 columns: 130 rows of 256 B, transposed layout [k][column]
        const float4* src4 = reinterpret_cast<const float4*>(a.lam + c0);
        float4* dst4 = reinterpret_cast<float4*>(lamS);
        for (int i = tid; i < OS_LAMW * 16; i += T)
            os_cp_async16(dst4 + i, src4 + (size_t)(i >> 4) * (Nx / 2) + (i & 15));
    }
    for (int i = tid; i < 129; i += T) csS[i] = __ldg(a.cs + i);
    for (int i = tid; i < 112; i += T) twS[i] = __ldg(a.tw + i);
    os_cp_async_commit_wait();
    __syncthreads();
    const int b = __float_as_int(lamS[129 * W + lane].x);
    const float ssh = lamS[129 * W + lane].y;
    const float* const col = a.src + c0 + lane;
    float* const ocol = a.dst + c0 + lane;

    const int ngroups = (nb + rb - 1) / rb;
    const int g0 = blockIdx.y * a.gpc, g1 = min(ngroups, g0 + a.gpc);
    auto land = [&](const int w, const int gi) {
        const int bl = w >> 4, t = w & 15, blk = gi * rb + bl;
        if (blk < nb)
            osv_land(reinterpret_cast<float*>(scr + (bl * MB + t) * W) + lane, col, Nx, vmask,
                     blk * OS_V - OS_H + b + 2 * t);
    };
    if (g0 < g1)
        for (int w = wid; w < rb * 16; w += nw) land(w, g0);
    for (int gi = g0; gi < g1; ++gi) {
        os_cp_async_commit_wait();                 // this thread's samples have landed
        // ---- pass A: scratch -> registers -> scratch, every thread on the slots it landed itself
#pragma unroll 1
        for (int w = wid; w < rb * 16; w += nw) {
            const int bl = w >> 4, t = w & 15;
            if (gi * rb + bl < nb)
                osv_fwd(reinterpret_cast<const float*>(scr + (bl * MB + t) * W) + lane, scr + (bl * MB + t) * W + lane,
                        twS + t);
        }
        __syncthreads();
        // ---- middle stage: item u of block bl, all 32 columns of the warp alike
#pragma unroll 1
        for (int w = wid; w < rb * 4; w += nw) {
            const int bl = w >> 2, u = w & 3;
            if (gi * rb + bl >= nb) continue;
            float2* const sb = scr + bl * MB * W + lane;
            if (u == 0) osv_mid<true>(sb, 0, lamS + lane, csS, dcS + bl * W + lane);
            else osv_mid<false>(sb, u, lamS + lane, csS, nullptr);
        }
        __syncthreads();
        // ---- inverse pass A: scratch -> registers -> global (+ delta-f source)
#pragma unroll 1
        for (int w = wid; w < rb * 16; w += nw) {
            const int bl = w >> 4, t = w & 15;
            const int blk = gi * rb + bl;
            if (blk >= nb) continue;
            const float2* o = scr + (bl * MB + t) * W + lane;
            float2 x[8];
            x[0] = o[0];
#pragma unroll
            for (int q = 1; q < 8; ++q) x[brev(q, 8)] = cmulc(o[q * 16 * W], twS[(q - 1) * 16 + t]);
            idft_dit<8, 1>(x);
            const float dc = dcS[bl * W + lane];
            const int row0 = blk * OS_V - OS_H + 2 * t;           // + 32 k, two rows per complex sample
            const float2 d2 = make_float2(dc, dc);
#pragma unroll
            for (int k = 0; k < 8; ++k) x[k] = cadd(x[k], d2);
            if (a.ng > 0) {                                       // delta-f source
                // f_eq,g(v - s) - f_eq,g(v) = f_eq,g(v) expm1(x_j),  x_j = c s (2 (v_j - mu) - s).  x_j is affine
                // in the row j, so along the rows of this thread expm1 obeys e' = e R + (R - 1): one expm1 per
                // item and two constants per row stride instead of one expm1 per cell (7 recurrence steps:
                // a few ulp of the source term).
#pragma unroll 1
                for (int g = 0; g < a.ng; ++g) {
                    const float cgs = a.cg4[g] * ssh;
                    const float* __restrict__ ft = a.feq_tab + g * Nv;
                    const float u0 = __ldg(a.vmu_tab + g * Nv);                // v_0 - mu_g
                    const float h1 = 2.0f * cgs * a.dvf, h32 = 32.0f * h1;
                    const float r1 = expm1f(h1);
                    const float R32 = expf(h32), r32 = expm1f(h32);
                    float ea = expm1f(cgs * (2.0f * fmaf((float)row0, a.dvf, u0) - ssh));
                    float eb = fmaf(ea, expf(h1), r1);
#pragma unroll
                    for (int k = 0; k < 8; ++k) {
                        const int j = min(max(row0 + 32 * k, 0), Nv - 2);     // rows outside are never stored
                        x[k].x = fmaf(__ldg(ft + j), ea, x[k].x);
                        x[k].y = fmaf(__ldg(ft + j + 1), eb, x[k].y);
                        ea = fmaf(ea, R32, r32);
                        eb = fmaf(eb, R32, r32);
                    }
                }
            }
            float* po = ocol + row0 * Nx;
            const int s32 = 32 * Nx;
#pragma unroll
            for (int k = 0; k < 8; ++k) {
                const int n = t + 16 * k;
                if (n >= osv::HN && n < osv::HN + osv::VN && row0 + 32 * k < Nv) {
                    __stcs(po, x[k].x);
                    __stcs(po + Nx, x[k].y);
                }
                po += s32;
            }
            if (gi + 1 < g1) land(w, gi + 1);      // the next group's item lands in the slots just read
        }
        // no barrier here: pass A touches only a thread's own slots, and dcS is rewritten only after the
        // barrier that follows the next pass A
    }
}

}  // namespace vog
