// vog_stencil.cu -- the circulant product of P:98-100 (eq (4)) taken DIRECTLY, u'_i = sum_j a_j u_{i+b+j}, instead of in
// Fourier space (the row of A has 2d+2 non-zeros for Lagrange 2d+1).  It is the same
// matrix as the Fourier path's up to rounding, selected per plan with vog_plan_tune(27, 1), for lines of >= 1024 cells;
// it is NOT the path BASELINE.json's north_star grades (that one is computed in Fourier space), it goes beside it:
// 2d+2 multiply-adds per cell beat the transform's instruction count, so these kernels sit on the memory roof.
// Product code; shares nothing with oracle/.
//
//   taps   : per line, the non-zero part of the first row of A, a_j, j = -JL .. JR, in fp64 -> fp32 (S1)
//              Lagrange 2d+1: a_j = prod_{k != j} (b* - k)/(j - k), j = -d .. d+1, padded with zeros to the
//                                     template's reach (NT = 4, 10 or 18 taps);
//              cubic spline: a = m * g, m = (B(b*+1), B(b*), B(b*-1), B(b*-2)) at j = -1..2 and
//                                     g_n = sqrt(3) (sqrt(3) - 2)^|n| the inverse of the collocation circulant
//                                     C(1/6, 4/6, 1/6); cut at |j| <= 14 like the Fourier path's blocks (reading Q6b:
//                                     the neglected part of the row sums to <= 8.4e-9 max|u|), NT = 29 taps.
//   x      : a half-warp owns a segment of 512 cells of a line; its window (512 + NT - 1 cells of the rolled line, 16-byte
//            aligned) and the taps row of its line land in one of its two slots by bulk asynchronous copies (the next
//            group's window is in flight in the other slot); a thread computes four consecutive cells at a time from
//            128-bit shared loads and stores them with one 128-bit store.  In place: a CTA-wide "landed" mbarrier
//            (as in osx7_kernel) before the first store of a line group; out of place: no synchronisation between warps.
//   v      : a CTA owns 32 columns x 128 rows; the union of the rows it needs lands coalesced in shared memory
//            (raw[row][column], conflict free for any per-column shift); a thread computes 16 consecutive rows of its
//            column from a sliding register window; rows are stored coalesced; the delta-f source is added in
//            the same pass.  Out of place, like the Fourier v kernels.
#include "vog_os2.cuh"

namespace vog {

// ---------------------------------------------------------------------------------------------
// S1 for the stencil path.  x: taps[line][32] (128-byte rows); v: taps[32][ks] transposed.  Entry 30 = s = E dt of the
// delta-f source (v), entry 31 = b mod N as int bits.
__global__ void __launch_bounds__(128) st_setup_kernel(const OsSetupArgs s, const int NT, const int JL, float* __restrict__ taps)
{
    const int l = blockIdx.x * blockDim.x + threadIdx.x;
    pdl_wait();                                   // E comes from the Poisson kernel; the tables may still be read
    pdl_launch_dependents();
    if (l >= s.n_lines) return;
    double beta;
    float sshift = 0.0f;
    if (s.mode == 0) {
        beta = -(s.vmin + (double)l * s.dv) * s.dt / s.delta;
    } else if (s.mode == 1) {
        double e = (double)s.E[l];
        if (s.Eext) e += (double)s.Eext[l];
        beta = -e * s.dt / s.delta;
        sshift = (float)(s.dt * e);
    } else {
        beta = s.beta[l];
    }
    const double fl = floor(beta);
    const double t = beta - fl;
    int b;
    if (fabs(fl) < 9.0e18) {                         // N is a power of two: mathematical mod by masking
        b = (int)(__double2ll_rn(fl) & (long long)(s.N - 1));
    } else {
        double bm = fmod(fl, (double)s.N);
        if (bm < 0.0) bm += (double)s.N;
        b = (int)bm;
        if (b >= s.N) b = 0;
    }
    float* out = s.vdir ? taps + l : taps + (size_t)l * 32;
    const size_t ks = s.vdir ? (size_t)s.ks : 1;
    for (int k = 0; k < 30; ++k) {
        const int j = k - JL;                        // tap index
        double a = 0.0;
        if (k < NT) {
            if (!s.spline) {
                if (j >= -s.d && j <= s.d + 1) {
                    a = 1.0;
                    for (int m = -s.d; m <= s.d + 1; ++m)
                        if (m != j) a *= (t - (double)m) / (double)(j - m);
                }
            } else {
                const double u = 1.0 - t;
                const double mq[4] = {u * u * u / 6.0, (4.0 - 6.0 * t * t + 3.0 * t * t * t) / 6.0,
                                      (1.0 + 3.0 * t + 3.0 * t * t - 3.0 * t * t * t) / 6.0, t * t * t / 6.0};   // j = -1..2
                const double rt3 = 1.7320508075688772935, q = rt3 - 2.0;    // g_n = sqrt(3) (sqrt(3) - 2)^|n|
                for (int p = 0; p < 4; ++p) {
                    const int n = j - (p - 1);
                    a += mq[p] * rt3 * pow(q, (double)(n < 0 ? -n : n));
                }
            }
        }
        out[k * ks] = (float)a;
    }
    out[30 * ks] = sshift;
    out[31 * ks] = __int_as_float(b);
}

// ---------------------------------------------------------------------------------------------
// x-direction
namespace st {
constexpr int SEG = 512;               // cells of a line per half-warp
__host__ __device__ constexpr int wcopy(int NT) { return (SEG + NT - 1 + 3 + 3) & ~3; }   // floats copied per window
__host__ __device__ constexpr int slotf(int NT) { return wcopy(NT) + 32; }                // + taps row (entry 31: integer shift)
}

// four consecutive outputs from the register window r (window offset M = misalignment of the first input, 0..3)
template <int NT, int M>
__device__ __forceinline__ float4 st_dot4(const float* r, const float* w)
{
    float a0 = 0.f, a1 = 0.f, a2 = 0.f, a3 = 0.f;
#pragma unroll
    for (int j = 0; j < NT; ++j) {
        a0 = fmaf(w[j], r[M + j], a0);
        a1 = fmaf(w[j], r[M + j + 1], a1);
        a2 = fmaf(w[j], r[M + j + 2], a2);
        a3 = fmaf(w[j], r[M + j + 3], a3);
    }
    return make_float4(a0, a1, a2, a3);
}

template <int NT, int JL, bool INPLACE>
__global__ void __launch_bounds__(512, 1) stx_kernel(const OsArgs a, const float* __restrict__ taps)
{
    extern __shared__ __align__(128) unsigned char smem_raw[];
    constexpr int WC = st::wcopy(NT), SF = st::slotf(NT);
    constexpr int L4 = (3 + NT + 3 + 3) / 4;       // 128-bit loads per four outputs
    const int lpi = a.lpi, ns = a.np;              // lines per group, segments per line
    const int nslot = lpi * ns;
    const int tid = threadIdx.x, T = blockDim.x, t = tid & 15, hw = tid >> 4, lane = tid & 31, warp = tid >> 5;
    const int N = a.N, mask = N - 1, nwarps = T >> 5;
    // two slots per half-warp (window | taps row | shift): the window of the NEXT group lands in the other slot while
    // this one is consumed
    float* const slot0 = reinterpret_cast<float*>(smem_raw) + hw * 2 * SF;
    unsigned long long* const bars = reinterpret_cast<unsigned long long*>(reinterpret_cast<float*>(smem_raw) + (T >> 4) * 2 * SF);
    // bars: [0] landed; [1 + warp] windows of the warp (one barrier per thread, see osx7_kernel)
    if (tid <= nwarps) {
        os2::mbar_init(bars + tid, tid == 0 ? (unsigned)nwarps : 2u);
        os2::mbar_init_fence();
    }
    __syncthreads();
    pdl_wait();
    pdl_launch_dependents();
    const bool has_seg = hw < nslot;
    const int l = has_seg ? hw / ns : 0, sg = hw - l * ns;     // line of the group, segment of the line
    const int G = gridDim.x;
    // leader of a half-warp: window, taps row (its entry 31 is the integer shift) of this segment in group g -> slot
    auto issue = [&](const int g, float* const win) {
        const int line = g * lpi + l;
        if (!has_seg || g >= a.n_groups || line >= a.n_lines) { os2::mbar_arrive(bars + 1 + warp); return; }
        const int b = __float_as_int(__ldg(taps + (size_t)line * 32 + 31));
        os2::mbar_expect_tx(bars + 1 + warp, 4u * WC + 128u);
        const float* const gl = a.src + (size_t)line * N;
        const int a0 = ((sg * st::SEG - JL + b) & mask) & ~3;
        if (a0 + WC <= N) os2::bulk_g2s(win, gl + a0, 4u * WC, bars + 1 + warp);
        else {
            const int n1 = N - a0;
            os2::bulk_g2s(win, gl + a0, 4u * (unsigned)n1, bars + 1 + warp);
            os2::bulk_g2s(win + n1, gl, 4u * (unsigned)(WC - n1), bars + 1 + warp);
        }
        os2::bulk_g2s(win + WC, taps + (size_t)line * 32, 128u, bars + 1 + warp);
    };
    if ((int)blockIdx.x < a.n_groups && t == 0) issue(blockIdx.x, slot0);
    unsigned parity = 0;
    for (int g = blockIdx.x; g < a.n_groups; g += G) {
        const int gn = g + G;
        const int line = g * lpi + l;
        const bool active = has_seg && line < a.n_lines;
        float* const win = slot0 + parity * SF;
        os2::mbar_wait(bars + 1 + warp, parity);   // this warp's windows have landed
        __syncwarp();                              // (every lane has seen this phase before the leaders arm the next one)
        // the other slot was consumed an iteration ago: the next group's window lands there during this iteration
        // (the shift it needs is a global load by the leader: one L2 latency per group, hidden by the other warps)
        if (t == 0 && gn < a.n_groups) issue(gn, slot0 + (parity ^ 1u) * SF);
        if (t == 0 && sg == 0 && has_seg && (gn + G) * lpi + l < a.n_lines)
            os2::bulk_prefetch_l2(a.src + (size_t)((gn + G) * lpi + l) * N, 4u * (unsigned)N);
        if constexpr (INPLACE) {
            // a store to a line may only be issued once every window of that line is on chip
            if (lane == 0) os2::mbar_arrive(bars);
            os2::mbar_wait(bars, parity);
        }
        if (active) {
            const float* const wrow = win + WC;
            float w[NT];
#pragma unroll
            for (int j = 0; j < NT; ++j) w[j] = wrow[j];
            const int m = ((sg * st::SEG - JL + __float_as_int(wrow[31])) & mask) & 3;       // uniform over the half-warp
            float4* const o4 = reinterpret_cast<float4*>(a.dst + (size_t)line * N + sg * st::SEG) + t;
#pragma unroll 2
            for (int k = 0; k < 8; ++k) {
                const float4* const p4 = reinterpret_cast<const float4*>(win) + t + 16 * k;
                float r[4 * L4];
#pragma unroll
                for (int i = 0; i < L4; ++i) {
                    const float4 v = p4[i];
                    r[4 * i] = v.x; r[4 * i + 1] = v.y; r[4 * i + 2] = v.z; r[4 * i + 3] = v.w;
                }
                float4 o;
                switch (m) {
                    case 0: o = st_dot4<NT, 0>(r, w); break;
                    case 1: o = st_dot4<NT, 1>(r, w); break;
                    case 2: o = st_dot4<NT, 2>(r, w); break;
                    default: o = st_dot4<NT, 3>(r, w); break;
                }
                __stcs(o4 + 16 * k, o);
            }
        }
        __syncwarp();
        parity ^= 1u;
    }
}

// ---------------------------------------------------------------------------------------------
// v-direction
namespace st {
constexpr int VRS = 128;               // rows per CTA (8 warps x 16 rows; four CTAs per SM interleave load, compute, store)
constexpr int VR = 16;                 // consecutive rows per thread
constexpr int VSPREAD = 32;            // spread of the integer shifts of a strip that the row buffer can hold
}

template <int NT, int JL>
__global__ void __launch_bounds__(256, 4) stv_kernel(const OsArgs a, const float* __restrict__ taps)
{
    extern __shared__ __align__(128) unsigned char smem_raw[];
    constexpr int W = 32, RS = st::VRS, R = st::VR, RMAX = st::VSPREAD;
    float* const raw = reinterpret_cast<float*>(smem_raw);                        // [RS + NT - 1 + RMAX][32]
    const int tid = threadIdx.x, lane = tid & 31, wid = tid >> 5;                 // column of the strip, row sub-segment
    const int Nx = a.Nx, Nv = a.Nv, vmask = Nv - 1;
    const int c0 = blockIdx.x * W, r0 = blockIdx.y * RS;
    const size_t ks = (size_t)a.lam_ks;
    pdl_wait();                                   // the taps and the source grid come from earlier kernels
    pdl_launch_dependents();
    const float* __restrict__ const tc = taps + c0 + lane;                        // entry k of this column: tc[k ks]
    float w[NT];
#pragma unroll
    for (int j = 0; j < NT; ++j) w[j] = __ldg(tc + j * ks);
    const float ssh = __ldg(tc + 30 * ks);
    const int b = __float_as_int(__ldg(tc + 31 * ks));
    // spread of the shifts over the strip, as signed distances from column 0's (shifts live mod Nv)
    const int b0 = __shfl_sync(0xffffffffu, b, 0);
    const int d = (((b - b0) + (Nv >> 1)) & vmask) - (Nv >> 1);
    int dmin = d, dmax = d;
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) {
        dmin = min(dmin, __shfl_xor_sync(0xffffffffu, dmin, o));
        dmax = max(dmax, __shfl_xor_sync(0xffffffffu, dmax, o));
    }
    const int Rs = dmax - dmin;
    const bool gather = Rs > RMAX;                 // uniform over the CTA
    const int db = gather ? 0 : d - dmin;          // this lane's row offset inside the raw rows
    const int base = gather ? b : b0 + dmin;       // first raw row = r0 - JL + base
    const int nrows = RS + NT - 1 + (gather ? 0 : Rs);
    const int rs = r0 - JL + base;
    if (!gather) {
        const float* const src = a.src + c0;
        for (int i = tid; i < nrows * 8; i += 256) {
            const int r = i >> 3, q4 = (i & 7) * 4;
            os2::cp_async16_cg(raw + r * W + q4, src + (size_t)((rs + r) & vmask) * Nx + q4);
        }
    } else {
        const float* const col = a.src + c0 + lane;
        for (int r = wid; r < nrows; r += 8) os2::cp_async4(raw + r * W + lane, col + (size_t)((rs + r) & vmask) * Nx);
    }
    os2::cp_async_wait_all();
    __syncthreads();
    // ---- 16 consecutive rows of this lane's column from a sliding register window
    const float* const rp = raw + (wid * R + db) * W + lane;
    float acc[R];
#pragma unroll
    for (int i = 0; i < R; ++i) acc[i] = 0.f;
#pragma unroll
    for (int k = 0; k < R + NT - 1; ++k) {         // input row k contributes to outputs i = k - j, j = tap index
        const float u = rp[k * W];
#pragma unroll
        for (int j = 0; j < NT; ++j) {
            const int i = k - j;
            if (i >= 0 && i < R) acc[i] = fmaf(w[j], u, acc[i]);
        }
    }
    const int row0 = r0 + wid * R;
    // ---- delta-f source: acc_i += f_eq,g(v_j) expm1(X_j), X_j = c s (2 (v_j - mu) - s) affine in the row j, so
    // expm1 obeys e' = e R + r along rows (R = exp(h), r = expm1(h), h = 2 c s dv); the recurrence starts in the middle
    // of the 16 rows and runs both ways, so at most 8 steps accumulate.
    if (a.ng > 0) {
#pragma unroll 1
        for (int g = 0; g < a.ng; ++g) {
            const float cgs = a.cg4[g] * ssh;
            const float* __restrict__ fa = a.feq_tab + g * Nv + row0;
            const float u0 = __ldg(a.vmu_tab + g * Nv);                          // v_0 - mu_g
            const float hh = 2.0f * cgs * a.dvf;
            const float Rf = expf(hh), rf = expm1f(hh), Rb = expf(-hh), rb = expm1f(-hh);
            const float e8 = expm1f(cgs * (2.0f * fmaf((float)(row0 + 8), a.dvf, u0) - ssh));
            float e = e8;
#pragma unroll
            for (int i = 8; i < R; ++i) {
                acc[i] = fmaf(__ldg(fa + i), e, acc[i]);
                e = fmaf(e, Rf, rf);
            }
            e = e8;
#pragma unroll
            for (int i = 7; i >= 0; --i) {
                e = fmaf(e, Rb, rb);
                acc[i] = fmaf(__ldg(fa + i), e, acc[i]);
            }
        }
    }
    float* const po = a.dst + (size_t)row0 * Nx + c0 + lane;
#pragma unroll
    for (int i = 0; i < R; ++i) __stcs(po + (size_t)i * Nx, acc[i]);
}

// ---------------------------------------------------------------------------------------------
// launchers.  tap template of a plan: Lagrange degree <= 3 -> (4, 1), <= 9 -> (10, 4), <= 17 -> (18, 8); spline -> (29, 14)
void st_template(int spline, int d, int* NT, int* JL)
{
    if (spline) { *NT = 29; *JL = 14; }
    else if (d <= 1) { *NT = 4; *JL = 1; }
    else if (d <= 4) { *NT = 10; *JL = 4; }
    else { *NT = 18; *JL = 8; }
}

cudaError_t st_setup_launch(const OsSetupArgs& s, float* taps, cudaStream_t st)
{
    int NT, JL;
    st_template(s.spline, s.d, &NT, &JL);
    return launch_pdl(st_setup_kernel, dim3((s.n_lines + 127) / 128), dim3(128), 0, st, s, NT, JL, taps);
}

size_t stx_smem_bytes(int spline, int d, int threads)
{
    int NT, JL;
    st_template(spline, d, &NT, &JL);
    return (size_t)(threads / 16) * 2 * st::slotf(NT) * 4 + (size_t)(threads / 32 + 1) * 8;
}

template <int NT, int JL>
static cudaError_t stx_launch_t(const OsArgs& a, const float* taps, int grid, int threads, size_t smem, cudaStream_t st)
{
    if (a.src == a.dst) {
        cudaError_t e = set_max_smem((const void*)stx_kernel<NT, JL, true>, smem);
        if (e != cudaSuccess) return e;
        return launch_pdl(stx_kernel<NT, JL, true>, dim3(grid), dim3(threads), smem, st, a, taps);
    }
    cudaError_t e = set_max_smem((const void*)stx_kernel<NT, JL, false>, smem);
    if (e != cudaSuccess) return e;
    return launch_pdl(stx_kernel<NT, JL, false>, dim3(grid), dim3(threads), smem, st, a, taps);
}

template <int NT, int JL>
static int stx_occ_t(int threads, size_t smem)
{
    if (set_max_smem((const void*)stx_kernel<NT, JL, true>, smem) != cudaSuccess) { cudaGetLastError(); return 0; }
    int nb = 0;
    if (cudaOccupancyMaxActiveBlocksPerMultiprocessor(&nb, stx_kernel<NT, JL, true>, threads, smem) != cudaSuccess) { cudaGetLastError(); return 0; }
    return nb;
}

cudaError_t stx_launch(const OsArgs& a, int spline, int d, const float* taps, int grid, int threads, size_t smem, cudaStream_t st)
{
    int NT, JL;
    st_template(spline, d, &NT, &JL);
    switch (NT) {
        case 4: return stx_launch_t<4, 1>(a, taps, grid, threads, smem, st);
        case 10: return stx_launch_t<10, 4>(a, taps, grid, threads, smem, st);
        case 18: return stx_launch_t<18, 8>(a, taps, grid, threads, smem, st);
        default: return stx_launch_t<29, 14>(a, taps, grid, threads, smem, st);
    }
}

int stx_occupancy(int spline, int d, int threads, size_t smem)
{
    int NT, JL;
    st_template(spline, d, &NT, &JL);
    switch (NT) {
        case 4: return stx_occ_t<4, 1>(threads, smem);
        case 10: return stx_occ_t<10, 4>(threads, smem);
        case 18: return stx_occ_t<18, 8>(threads, smem);
        default: return stx_occ_t<29, 14>(threads, smem);
    }
}

template <int NT, int JL>
static cudaError_t stv_launch_t(const OsArgs& a, const float* taps, cudaStream_t st)
{
    const size_t smem = (size_t)(st::VRS + NT - 1 + st::VSPREAD) * 32 * 4;
    cudaError_t e = set_max_smem((const void*)stv_kernel<NT, JL>, smem);
    if (e != cudaSuccess) return e;
    return launch_pdl(stv_kernel<NT, JL>, dim3(a.Nx / 32, a.Nv / st::VRS), dim3(256), smem, st, a, taps);
}

cudaError_t stv_launch(const OsArgs& a, int spline, int d, const float* taps, cudaStream_t st)
{
    int NT, JL;
    st_template(spline, d, &NT, &JL);
    switch (NT) {
        case 4: return stv_launch_t<4, 1>(a, taps, st);
        case 10: return stv_launch_t<10, 4>(a, taps, st);
        case 18: return stv_launch_t<18, 8>(a, taps, st);
        default: return stv_launch_t<29, 14>(a, taps, st);
    }
}

}  // namespace vog
