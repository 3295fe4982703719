// vog_f64.cu -- double-precision mode ("generally a factor of two": the
// long-time runs that single precision cannot follow).  The whole path once more with f, rho, E and every table in
// fp64: the circulant product of eq (4) taken in its direct form u'_i = sum_j a_j u_{i+b+j} (the row of A has
// 2d+2 non-zeros for Lagrange 2d+1; for the cubic spline a = m * g with g_n = sqrt(3) (sqrt(3) - 2)^|n| cut at
// |n| <= 30, where the neglected part of the row is below 1e-17), the density by fixed-order column sums, the field by
// the Fourier solve of P:221 written as two plain DFT sums spread over the GPU (O(Nx^2) multiply-adds: 0.3 % of the
// step's time at 2048^2 and under 10 % at 16384^2, exact to rounding, no fp64 FFT to maintain), the delta-f source of
// P:197 with expm1 in fp64.  Why the direct form here and not transforms: in fp64 the B200 issues 64 multiply-adds per
// SM and clock, 18 taps are 65 us of arithmetic per 8192^2 advection against 164 us of memory traffic at 16 B per cell:
// the kernels below are memory-bound without a transform, so the transform would only add rounding.
// Product code; shares nothing with oracle/.
#include <cuda_runtime.h>

#include <cmath>
#include <new>

#include "vog_os2.cuh"

namespace vog {

namespace f64 {
constexpr int NTMAX = 64;              // taps per line (Lagrange: order + 1; cubic spline: 64)
constexpr int NBY = 8;                 // density row slabs
}

struct F64SetupArgs {
    int n_lines, N, mode;      // mode 0: beta = -v_l dt / dx; 1: beta = -(E_l + Eext_l) dt / dv; 2: explicit beta
    int spline, d, NT, JL;     // taps j = -JL .. NT - 1 - JL
    long long ls, ks;          // taps[l * ls + k * ks]
    double dt, delta, vmin, dv;
    const double* E;
    const double* Eext;
    const double* beta;
};

// S1 in fp64: integer shift b, taps a_j of the first row of A, and (v direction) the source shift s = E dt.
// One thread per (line, tap): with one thread per line the 2d+2 products of 2d+1 factors ran one after the other in
// every thread (33 us for 2048 lines, a quarter of the 2048^2 step).
__global__ void __launch_bounds__(128) f64_setup_kernel(const F64SetupArgs s, double* __restrict__ taps, int* __restrict__ bsh,
                                                        double* __restrict__ ssh)
{
    const long long idx = (long long)blockIdx.x * blockDim.x + threadIdx.x;
    const int l = (int)(idx / s.NT), k = (int)(idx - (long long)l * s.NT);
    if (l >= s.n_lines) return;
    double beta, sshift = 0.0;
    if (s.mode == 0) {
        beta = -(s.vmin + (double)l * s.dv) * s.dt / s.delta;
    } else if (s.mode == 1) {
        double e = s.E[l];
        if (s.Eext) e += s.Eext[l];
        beta = -e * s.dt / s.delta;
        sshift = s.dt * e;
    } else {
        beta = s.beta[l];
    }
    const double fl = floor(beta);
    const double t = beta - fl;                      // b* in [0, 1)
    double* const out = taps + (long long)l * s.ls;
    if (k == 0) {
        int b;
        if (fabs(fl) < 9.0e18) {                     // N is a power of two: mathematical mod by masking
            b = (int)(__double2ll_rn(fl) & (long long)(s.N - 1));
        } else {
            double bm = fmod(fl, (double)s.N);
            if (bm < 0.0) bm += (double)s.N;
            b = (int)bm;
            if (b >= s.N) b = 0;
        }
        bsh[l] = b;
        if (ssh) ssh[l] = sshift;
        if (s.ks == 1) { out[s.NT] = (double)b; out[s.NT + 1] = 0.0; }       // x rows: (taps, b, pad), see f64_x_kernel
    }
    const int j = k - s.JL;
    double a = 0.0;
    if (!s.spline) {
        // Lagrange 2d+1: a_j = prod_{m != j} (b* - m) / (j - m), j = -d .. d+1 (zero outside: the kernels
        // are compiled for 4, 10 and 18 taps).  The denominator is an integer of at most 17! < 2^53: exact.
        if (j >= -s.d && j <= s.d + 1) {
            double num = 1.0, den = 1.0;
            for (int m = -s.d; m <= s.d + 1; ++m)
                if (m != j) { num *= t - (double)m; den *= (double)(j - m); }
            a = num / den;
        }
    } else {
        // cubic spline: a = m * g, m = (B(b*+1), B(b*), B(b*-1), B(b*-2)) at j = -1..2
        const double u = 1.0 - t;
        const double mq[4] = {u * u * u / 6.0, (4.0 - 6.0 * t * t + 3.0 * t * t * t) / 6.0,
                              (1.0 + 3.0 * t + 3.0 * t * t - 3.0 * t * t * t) / 6.0, t * t * t / 6.0};
        const double rt3 = 1.7320508075688772935, q = rt3 - 2.0;
        for (int p = 0; p < 4; ++p) {
            const int n = j - (p - 1);
            a += mq[p] * rt3 * pow(q, (double)(n < 0 ? -n : n));
        }
    }
    out[k * s.ks] = a;
}

// ---------------------------------------------------------------------------------------------
// x direction: a persistent CTA owns whole lines.  One thread lands the NEXT line and its row of taps in shared memory
// with bulk asynchronous copies (cp.async.bulk, completion counted in bytes on an mbarrier) while the CTA computes the
// current one from the other buffer (two buffers when 2 Nx doubles fit, one for 16384-cell lines).  The whole line is on
// chip before its first store: in place needs no further care.
// Taps row of a line: NT doubles, then the integer shift b as a double, then one unused double (16-byte multiple).
//
// Two consecutive cells per thread from 128-bit shared loads: a warp reads 512 contiguous bytes per instruction, the
// conflict-free minimum of four wavefronts (four cells per thread from 64-bit loads put the lanes 32 bytes apart:
// eight wavefronts per load, and the kernel ran at the speed of the shared-memory pipe, 2.3 times slower).  be = the
// even base of the window, M = 1 when the first sample wanted is the odd one of its pair.
template <int NT, int M>
__device__ __forceinline__ void f64_x_cells(const double* __restrict__ line, const double* a, double* o, const int be,
                                            const int tid, const int T, const int Nx)
{
    constexpr int NL = (NT + 1 + M + 1) / 2;       // 128-bit loads for NT + 1 samples starting at offset M
    const int mask = Nx - 1;
    for (int i0 = 2 * tid; i0 < Nx; i0 += 2 * T) {
        double r[2 * NL];
#pragma unroll
        for (int n = 0; n < NL; ++n) {
            const double2 v = *reinterpret_cast<const double2*>(line + ((i0 + be + 2 * n) & mask));
            r[2 * n] = v.x;
            r[2 * n + 1] = v.y;
        }
        double acc0 = 0.0, acc1 = 0.0;
#pragma unroll
        for (int k = 0; k < NT; ++k) {
            acc0 = fma(a[k], r[M + k], acc0);
            acc1 = fma(a[k], r[M + k + 1], acc1);
        }
        *reinterpret_cast<double2*>(o + i0) = make_double2(acc0, acc1);
    }
}

template <int NT>
__global__ void __launch_bounds__(1024) f64_x_kernel(const double* src, double* dst, const int Nx, const int Nv,
                                                     const int nt_rt, const int JL, const int nbuf,
                                                     const double* __restrict__ taps)
{
    extern __shared__ __align__(128) unsigned char smem_raw[];
    const int nt = NT > 0 ? NT : nt_rt, tw = nt + 2;
    double* const lines = reinterpret_cast<double*>(smem_raw);                     // [nbuf][Nx]
    double* const tps = lines + (size_t)nbuf * Nx;                                 // [nbuf][tw]
    unsigned long long* const bars = reinterpret_cast<unsigned long long*>(tps + nbuf * f64::NTMAX + 2 * nbuf);
    const int tid = threadIdx.x, T = blockDim.x, mask = Nx - 1, G = gridDim.x;
    if (tid < nbuf) {                              // (one barrier per thread, see osx7_kernel)
        os2::mbar_init(bars + tid, 1u);
        os2::mbar_init_fence();
    }
    __syncthreads();
    auto request = [&](const int l, const int buf) {
        os2::mbar_expect_tx(bars + buf, (unsigned)(Nx * 8 + tw * 8));
        os2::bulk_g2s(lines + (size_t)buf * Nx, src + (size_t)l * Nx, (unsigned)Nx * 8u, bars + buf);
        os2::bulk_g2s(tps + buf * (f64::NTMAX + 2), taps + (size_t)l * tw, (unsigned)tw * 8u, bars + buf);
    };
    if (tid == 0 && blockIdx.x < Nv) request(blockIdx.x, 0);
    unsigned ph0 = 0, ph1 = 0;
    int it = 0;
    for (int l = blockIdx.x; l < Nv; l += G, ++it) {
        const int buf = nbuf == 2 ? (it & 1) : 0;
        if (nbuf == 2 && tid == 0 && l + G < Nv) request(l + G, buf ^ 1);          // (that buffer was released by the
                                                                                   // barrier that ended iteration it-1)
        if (buf == 0) { os2::mbar_wait(bars, ph0); ph0 ^= 1u; }
        else { os2::mbar_wait(bars + 1, ph1); ph1 ^= 1u; }
        const double* const line = lines + (size_t)buf * Nx;
        const double* const tp = tps + buf * (f64::NTMAX + 2);
        const int b = (int)tp[nt] - JL;
        double* const o = dst + (size_t)l * Nx;
        if constexpr (NT > 0) {
            double a[NT];
#pragma unroll
            for (int k = 0; k < NT; ++k) a[k] = tp[k];
            if (b & 1) f64_x_cells<NT, 1>(line, a, o, b - 1, tid, T, Nx);
            else f64_x_cells<NT, 0>(line, a, o, b, tid, T, Nx);
        } else {
            for (int i = tid; i < Nx; i += T) {
                double acc = 0.0;
                for (int k = 0; k < nt; ++k) acc = fma(tp[k], line[(i + b + k) & mask], acc);
                o[i] = acc;
            }
        }
        __syncthreads();                           // the line has been read by everybody: its buffer may be refilled
        if (nbuf == 1 && tid == 0 && l + G < Nv) request(l + G, 0);
    }
}

// ---------------------------------------------------------------------------------------------
// v direction, out of place: a thread owns a column and R = 16 consecutive rows; the rows it needs are read straight
// from global memory (neighbouring columns with the same integer shift read the same 256-byte row segments).  delta-f source: f_eq,g(v_j) expm1(c_g s (2 (v_j -
// mu_g) - s)) with s = E dt, summed over the Gaussians: f_eq(v - s) - f_eq(v) without the cancellation.
struct F64Feq { int n; double amp[4], mu[4], c[4]; };

template <int NT>
__global__ void __launch_bounds__(256) f64_v_kernel(const double* __restrict__ src, double* __restrict__ dst, const int Nx,
                                                    const int Nv, const int nt_rt, const int JL,
                                                    const double* __restrict__ taps, const int* __restrict__ bsh,
                                                    const double* __restrict__ ssh, const F64Feq fq, const double vmin,
                                                    const double dv)
{
    constexpr int R = 16;
    // block = 32 columns x (blockDim.x / 32) warps, warp w takes rows r0 .. r0 + 15 of the block's row range: the
    // NT - 1 rows a warp shares with the warp below it are hits in L1 (the loads go through the read-only path)
    const int c = blockIdx.x * 32 + (threadIdx.x & 31), mask = Nv - 1;
    const int r0 = (blockIdx.y * (blockDim.x >> 5) + (threadIdx.x >> 5)) * R;
    const int nt = NT > 0 ? NT : nt_rt;
    const int b = bsh[c] - JL;
    const double* const col = src + c;
    double acc[R];
#pragma unroll
    for (int r = 0; r < R; ++r) acc[r] = 0.0;
    if constexpr (NT > 0) {
        double a[NT];
#pragma unroll
        for (int k = 0; k < NT; ++k) a[k] = __ldg(taps + (size_t)k * Nx + c);
#pragma unroll
        for (int n = 0; n < NT + R - 1; ++n) {
            const double v = __ldg(col + (size_t)((r0 + b + n) & mask) * Nx);
#pragma unroll
            for (int r = 0; r < R; ++r)
                if (n - r >= 0 && n - r < NT) acc[r] = fma(a[n - r], v, acc[r]);
        }
    } else {
        for (int k = 0; k < nt; ++k) {
            const double ak = __ldg(taps + (size_t)k * Nx + c);
#pragma unroll
            for (int r = 0; r < R; ++r) acc[r] = fma(ak, __ldg(col + (size_t)((r0 + r + b + k) & mask) * Nx), acc[r]);
        }
    }
    if (fq.n > 0) {
        const double s = ssh[c];
#pragma unroll
        for (int r = 0; r < R; ++r) {
            const double v = vmin + (double)(r0 + r) * dv;
            double q = 0.0;
#pragma unroll
            for (int g = 0; g < 4; ++g) {
                if (g < fq.n) {
                    const double u = v - fq.mu[g];
                    q += fq.amp[g] * exp(-fq.c[g] * u * u) * expm1(fq.c[g] * s * (2.0 * u - s));
                }
            }
            acc[r] += q;
        }
    }
#pragma unroll
    for (int r = 0; r < R; ++r) dst[(size_t)(r0 + r) * Nx + c] = acc[r];
}

// ---------------------------------------------------------------------------------------------
// S8 in fp64: column sums of a row slab, fixed order.  grid (Nx / 64, NBY), 256 threads = 4 row lanes x 64 columns.
__global__ void __launch_bounds__(256) f64_density_kernel(const double* __restrict__ f, const int Nx, const int rows_per_block,
                                                          double* __restrict__ part)
{
    __shared__ double red[4][64];
    const int cl = threadIdx.x & 63, rl = threadIdx.x >> 6;
    const int col = blockIdx.x * 64 + cl;
    const int j0 = blockIdx.y * rows_per_block;
    double s = 0.0;
    const double* p = f + (size_t)(j0 + rl) * Nx + col;
#pragma unroll 8
    for (int j = rl; j < rows_per_block; j += 4) {
        s += __ldg(p);
        p += (size_t)4 * Nx;
    }
    red[rl][cl] = s;
    __syncthreads();
    if (rl == 0) part[(size_t)blockIdx.y * Nx + col] = ((red[0][cl] + red[1][cl]) + red[2][cl]) + red[3][cl];
}

// rho_i = dv * (slab sums in slab order); rt_i = rho_i - mean.  One CTA.
__global__ void __launch_bounds__(1024) f64_rho_kernel(const int Nx, const int nby, const double dv,
                                                       const double* __restrict__ part, double* __restrict__ rho,
                                                       double* __restrict__ rt)
{
    __shared__ double red[32];
    __shared__ double mean_s;
    const int tid = threadIdx.x, T = blockDim.x;
    double loc = 0.0;
    for (int i = tid; i < Nx; i += T) {
        double s = 0.0;
        for (int y = 0; y < nby; ++y) s += part[(size_t)y * Nx + i];
        s *= dv;
        rho[i] = s;
        loc += s;
    }
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) loc += __shfl_xor_sync(0xffffffffu, loc, o);
    if ((tid & 31) == 0) red[tid >> 5] = loc;
    __syncthreads();
    if (tid == 0) {
        double s = 0.0;
        for (int w = 0; w < (T + 31) / 32; ++w) s += red[w];
        mean_s = s / (double)Nx;
    }
    __syncthreads();
    const double mean = mean_s;
    for (int i = tid; i < Nx; i += T) rt[i] = rho[i] - mean;
}

// S9 in fp64, the Fourier solve of P:221 as two plain DFT sums.  tw[q] = (cos, sin)(2 pi q / Nx).
//   forward, one CTA of 128 threads per mode m = 1 .. Nx/2 - 1:  rho^_m = sum_i rt_i e^{-2 i pi m i / Nx};
//   E^_m = rho^_m / (i k_m), k_m = 2 pi m / L.  Modes 0 and Nx/2 are dropped (reading Q12).
//   Sums in a fixed order (thread-strided partial sums, shuffle tree, the four warps in order): deterministic.
__device__ __forceinline__ double2 f64_block_sum(double a, double b, double2* red)
{
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) {
        a += __shfl_xor_sync(0xffffffffu, a, o);
        b += __shfl_xor_sync(0xffffffffu, b, o);
    }
    if ((threadIdx.x & 31) == 0) red[threadIdx.x >> 5] = make_double2(a, b);
    __syncthreads();
    double2 s = red[0];
    for (int w = 1; w < (int)(blockDim.x >> 5); ++w) { s.x += red[w].x; s.y += red[w].y; }
    return s;
}

// The root of a term is the product of two table entries, e^{-2 i pi m i / Nx} with i = i1 + 128 i2: the first factor
// is the thread's own (loaded once), the second the same for the whole CTA (one broadcast load per term) -- a gather
// of tw[(m i) mod Nx] per term made these two kernels 18 % of the 8192^2 step.
__global__ void __launch_bounds__(128) f64_dft_fwd_kernel(const int Nx, const double L, const double* __restrict__ rt,
                                                          const double2* __restrict__ tw, double2* __restrict__ Ehat)
{
    __shared__ double2 red[4];
    const int m = 1 + blockIdx.x, mask = Nx - 1, T = blockDim.x;
    const double2 w1 = __ldg(tw + (int)(((long long)m * threadIdx.x) & mask));
    double sr = 0.0, si = 0.0;
    for (int i2 = 0; i2 * T < Nx; ++i2) {
        const double2 w2 = __ldg(tw + (int)(((long long)m * T * i2) & mask));
        const double wx = w1.x * w2.x - w1.y * w2.y, wy = w1.x * w2.y + w1.y * w2.x;
        const double r = rt[i2 * T + threadIdx.x];
        sr = fma(r, wx, sr);
        si = fma(-r, wy, si);
    }
    const double2 s = f64_block_sum(sr, si, red);
    if (threadIdx.x == 0) {
        const double k = 2.0 * 3.14159265358979323846 * (double)m / L;
        Ehat[m] = make_double2(s.y / k, -s.x / k);   // (sr + i si) / (i k)
    }
}

//   inverse, one CTA per cell i:  E_i = (1/Nx) sum_m E^_m e^{+2 i pi m i / Nx} = (2/Nx) sum_{0 < m < Nx/2} Re(..)
//   (E^_{Nx-m} is the conjugate of E^_m: rho is real); m = m1 + 128 m2 factored the same way.
__global__ void __launch_bounds__(128) f64_dft_inv_kernel(const int Nx, const double2* __restrict__ Ehat,
                                                          const double2* __restrict__ tw, double* __restrict__ E_a,
                                                          double* __restrict__ E_b)
{
    __shared__ double2 red[4];
    const int i = blockIdx.x, mask = Nx - 1, T = blockDim.x;
    const double2 w1 = __ldg(tw + (int)(((long long)threadIdx.x * i) & mask));
    double s = 0.0;
    for (int m2 = 0; m2 * T < Nx / 2; ++m2) {
        const int m = m2 * T + threadIdx.x;
        const double2 w2 = __ldg(tw + (int)(((long long)m2 * T * i) & mask));
        const double wx = w1.x * w2.x - w1.y * w2.y, wy = w1.x * w2.y + w1.y * w2.x;
        const double2 e = m >= 1 ? Ehat[m] : make_double2(0.0, 0.0);
        s += e.x * wx - e.y * wy;
    }
    const double2 t = f64_block_sum(s, 0.0, red);
    if (threadIdx.x == 0) {
        const double v = 2.0 * t.x / (double)Nx;
        E_a[i] = v;
        if (E_b) E_b[i] = v;
    }
}

__global__ void f64_tw_kernel(const int Nx, double2* __restrict__ tw)
{
    const int q = blockIdx.x * blockDim.x + threadIdx.x;
    if (q >= Nx) return;
    double sn, cs;
    sincospi(2.0 * (double)q / (double)Nx, &sn, &cs);
    tw[q] = make_double2(cs, sn);
}

__global__ void f64_add_kernel(const int n, const double* __restrict__ a, const double* __restrict__ b, double* __restrict__ o)
{
    const int i = blockIdx.x * blockDim.x + threadIdx.x;
    if (i < n) o[i] = a[i] + (b ? b[i] : 0.0);
}

// ==========================================================================================
// host side: the state of the fp64 mode of one plan (created on the first *_f64 call)
struct F64State {
    vog_params_t p;
    cudaStream_t st;
    int n_sm, NT, JL, d, spline;
    double *taps_x, *taps_v, *ssh_v;           // [Nv][NT]; [NT][Nx]; [Nx]
    int *b_x, *b_v;
    double *part, *rho, *rt, *E, *Et;          // slab sums [NBY][Nx]; rho; rho - mean; E; E + E_ext
    double2 *tw, *Ehat;
    double* g;                                 // second grid (out-of-place v-advection), allocated on first use
    bool x_valid, E_valid;
    double x_dt;
    const double* E_of;
    long long launches;
};

void f64_destroy(F64State* S);

static cudaError_t f64_setup(F64State* S, bool vdir, int mode, double dt, const double* E, const double* Eext, const double* beta)
{
    const int Nx = S->p.Nx, Nv = S->p.Nv;
    F64SetupArgs a;
    a.n_lines = vdir ? Nx : Nv;
    a.N = vdir ? Nv : Nx;
    a.mode = mode;
    a.spline = S->spline; a.d = S->d; a.NT = S->NT; a.JL = S->JL;
    a.ls = vdir ? 1 : S->NT + 2;
    a.ks = vdir ? Nx : 1;
    a.dt = dt;
    a.dv = (S->p.vmax - S->p.vmin) / (double)Nv;
    a.delta = vdir ? a.dv : S->p.L / (double)Nx;
    a.vmin = S->p.vmin;
    a.E = E; a.Eext = Eext; a.beta = beta;
    f64_setup_kernel<<<(unsigned)(((long long)a.n_lines * a.NT + 127) / 128), 128, 0, S->st>>>(a, vdir ? S->taps_v : S->taps_x, vdir ? S->b_v : S->b_x,
                                                                  vdir ? S->ssh_v : nullptr);
    S->launches++;
    return cudaGetLastError();
}

template <int NT>
static cudaError_t f64_x_launch_t(F64State* S, const double* src, double* dst)
{
    const int Nx = S->p.Nx, Nv = S->p.Nv;
    const int nbuf = Nx <= 8192 ? 2 : 1;
    const size_t smem = sizeof(double) * ((size_t)nbuf * Nx + nbuf * (f64::NTMAX + 2) + 2 * nbuf) + 16;
    cudaError_t e = set_max_smem((const void*)f64_x_kernel<NT>, smem);
    if (e != cudaSuccess) return e;
    int threads = NT > 0 ? Nx / 2 : Nx;
    if (threads > 1024) threads = 1024;
    if (threads < 64) threads = 64;
    int per_sm = (int)((220 * 1024) / (smem + 1024));
    if (per_sm > 2048 / threads) per_sm = 2048 / threads;
    if (per_sm < 1) per_sm = 1;
    int grid = S->n_sm * per_sm;
    if (grid > Nv) grid = Nv;
    f64_x_kernel<NT><<<grid, threads, smem, S->st>>>(src, dst, Nx, Nv, S->NT, S->JL, nbuf, S->taps_x);
    S->launches++;
    return cudaGetLastError();
}

static cudaError_t f64_x_launch(F64State* S, const double* src, double* dst)
{
    if (S->spline) return f64_x_launch_t<0>(S, src, dst);
    if (S->NT == 4) return f64_x_launch_t<4>(S, src, dst);
    if (S->NT == 10) return f64_x_launch_t<10>(S, src, dst);
    return f64_x_launch_t<18>(S, src, dst);
}

static cudaError_t f64_v_launch(F64State* S, const double* src, double* dst, bool source)
{
    const int Nx = S->p.Nx, Nv = S->p.Nv;
    F64Feq fq;
    fq.n = source ? S->p.feq.n : 0;
    for (int g = 0; g < 4; ++g) { fq.amp[g] = S->p.feq.amp[g]; fq.mu[g] = S->p.feq.mu[g]; fq.c[g] = S->p.feq.c[g]; }
    const double dv = (S->p.vmax - S->p.vmin) / (double)Nv;
    int warps = Nv / 16;                           // row groups of 16 per block (Nv >= 64: at least 4)
    if (warps > 8) warps = 8;
    const int threads = 32 * warps;
    const dim3 grid(Nx / 32, Nv / (16 * warps));
    if (S->spline) f64_v_kernel<0><<<grid, threads, 0, S->st>>>(src, dst, Nx, Nv, S->NT, S->JL, S->taps_v, S->b_v, S->ssh_v, fq, S->p.vmin, dv);
    else if (S->NT == 4) f64_v_kernel<4><<<grid, threads, 0, S->st>>>(src, dst, Nx, Nv, S->NT, S->JL, S->taps_v, S->b_v, S->ssh_v, fq, S->p.vmin, dv);
    else if (S->NT == 10) f64_v_kernel<10><<<grid, threads, 0, S->st>>>(src, dst, Nx, Nv, S->NT, S->JL, S->taps_v, S->b_v, S->ssh_v, fq, S->p.vmin, dv);
    else f64_v_kernel<18><<<grid, threads, 0, S->st>>>(src, dst, Nx, Nv, S->NT, S->JL, S->taps_v, S->b_v, S->ssh_v, fq, S->p.vmin, dv);
    S->launches++;
    return cudaGetLastError();
}

static cudaError_t f64_ensure_g(F64State* S)
{
    if (S->g) return cudaSuccess;
    return cudaMalloc((void**)&S->g, sizeof(double) * (size_t)S->p.Nx * S->p.Nv);
}

int f64_create(F64State** out, const vog_params_t* p, cudaStream_t st, int n_sm)
{
    F64State* S = new (std::nothrow) F64State();
    if (!S) return VOG_ENOMEM;
    S->p = *p; S->st = st; S->n_sm = n_sm;
    S->spline = p->kind == VOG_BSPLINE;
    S->d = S->spline ? 0 : (p->order - 1) / 2;
    if (S->spline) { S->NT = 64; S->JL = 31; }
    else if (p->order <= 3) { S->NT = 4; S->JL = 1; }
    else if (p->order <= 9) { S->NT = 10; S->JL = 4; }
    else { S->NT = 18; S->JL = 8; }
    const size_t Nx = p->Nx, Nv = p->Nv;
    cudaError_t e = cudaSuccess;
    auto alloc = [&](void** q, size_t bytes) { if (e == cudaSuccess) e = cudaMalloc(q, bytes); };
    alloc((void**)&S->taps_x, sizeof(double) * Nv * (S->NT + 2));
    alloc((void**)&S->taps_v, sizeof(double) * Nx * S->NT);
    alloc((void**)&S->ssh_v, sizeof(double) * Nx);
    alloc((void**)&S->b_x, sizeof(int) * Nv);
    alloc((void**)&S->b_v, sizeof(int) * Nx);
    alloc((void**)&S->part, sizeof(double) * f64::NBY * Nx);
    alloc((void**)&S->rho, sizeof(double) * Nx);
    alloc((void**)&S->rt, sizeof(double) * Nx);
    alloc((void**)&S->E, sizeof(double) * Nx);
    alloc((void**)&S->Et, sizeof(double) * Nx);
    alloc((void**)&S->tw, sizeof(double2) * Nx);
    alloc((void**)&S->Ehat, sizeof(double2) * Nx);
    if (e != cudaSuccess) { cudaGetLastError(); f64_destroy(S); return VOG_ENOMEM; }
    f64_tw_kernel<<<(p->Nx + 255) / 256, 256, 0, st>>>(p->Nx, S->tw);
    if (cudaGetLastError() != cudaSuccess) { f64_destroy(S); return VOG_ECUDA; }
    *out = S;
    return VOG_OK;
}

void f64_destroy(F64State* S)
{
    if (!S) return;
    cudaFree(S->taps_x); cudaFree(S->taps_v); cudaFree(S->ssh_v); cudaFree(S->b_x); cudaFree(S->b_v); cudaFree(S->part);
    cudaFree(S->rho); cudaFree(S->rt); cudaFree(S->E); cudaFree(S->Et); cudaFree(S->tw); cudaFree(S->Ehat); cudaFree(S->g);
    delete S;
}

long long f64_launches(const F64State* S) { return S ? S->launches : 0; }

cudaError_t f64_shift(F64State* S, double* f, const double* beta, bool vdir)
{
    S->x_valid = false; S->E_valid = false;
    cudaError_t e = f64_setup(S, vdir, 2, 0.0, nullptr, nullptr, beta);
    if (e != cudaSuccess) return e;
    if (!vdir) return f64_x_launch(S, f, f);
    e = f64_ensure_g(S);
    if (e == cudaSuccess) e = f64_v_launch(S, f, S->g, false);
    if (e == cudaSuccess) e = cudaMemcpyAsync(f, S->g, sizeof(double) * (size_t)S->p.Nx * S->p.Nv, cudaMemcpyDeviceToDevice, S->st);
    return e;
}

static cudaError_t f64_x(F64State* S, const double* src, double* dst, double dt)
{
    if (!(S->x_valid && S->x_dt == dt)) {
        cudaError_t e = f64_setup(S, false, 0, dt, nullptr, nullptr, nullptr);
        if (e != cudaSuccess) return e;
        S->x_valid = true; S->x_dt = dt;
    }
    return f64_x_launch(S, src, dst);
}

cudaError_t f64_advect_x(F64State* S, double* f, double dt)
{
    S->E_valid = false;
    return f64_x(S, f, f, dt);
}

cudaError_t f64_advect_v(F64State* S, double* f, const double* E, double dt)
{
    S->E_valid = false;
    cudaError_t e = f64_setup(S, true, 1, dt, E, nullptr, nullptr);
    if (e == cudaSuccess) e = f64_ensure_g(S);
    if (e == cudaSuccess) e = f64_v_launch(S, f, S->g, true);
    if (e == cudaSuccess) e = cudaMemcpyAsync(f, S->g, sizeof(double) * (size_t)S->p.Nx * S->p.Nv, cudaMemcpyDeviceToDevice, S->st);
    return e;
}

// density + Fourier solve of f into S->E (and E_out)
cudaError_t f64_field(F64State* S, const double* f, double* E_out)
{
    const int Nx = S->p.Nx, Nv = S->p.Nv;
    const double dv = (S->p.vmax - S->p.vmin) / (double)Nv;
    int nby = f64::NBY;
    while (nby > 1 && Nv / nby < 16) nby >>= 1;
    f64_density_kernel<<<dim3(Nx / 64, nby), 256, 0, S->st>>>(f, Nx, Nv / nby, S->part);
    f64_rho_kernel<<<1, Nx < 1024 ? Nx : 1024, 0, S->st>>>(Nx, nby, dv, S->part, S->rho, S->rt);
    const int dft_threads = Nx / 2 < 128 ? Nx / 2 : 128;   // divides Nx / 2
    f64_dft_fwd_kernel<<<Nx / 2 - 1, dft_threads, 0, S->st>>>(Nx, S->p.L, S->rt, S->tw, S->Ehat);
    f64_dft_inv_kernel<<<Nx, dft_threads, 0, S->st>>>(Nx, S->Ehat, S->tw, S->E, E_out);
    S->launches += 4;
    S->E_valid = true;
    S->E_of = f;
    return cudaGetLastError();
}

cudaError_t f64_get_field(F64State* S, double* E)
{
    return cudaMemcpyAsync(E, S->E, sizeof(double) * S->p.Nx, cudaMemcpyDeviceToDevice, S->st);
}

bool f64_has_field(const F64State* S) { return S && S->E_valid; }

static cudaError_t f64_v_total(F64State* S, const double* src, double* dst, double dt, const double* Eext)
{
    cudaError_t e = f64_setup(S, true, 1, dt, S->E, Eext, nullptr);
    if (e == cudaSuccess) e = f64_v_launch(S, src, dst, true);
    return e;
}

// One Strang step, the sequences of vog_step; the v-advection writes the second grid and the following
// x-advection reads it back, so no copy is made.
cudaError_t f64_step(F64State* S, double* f, double dt, const double* Eext)
{
    cudaError_t e = f64_ensure_g(S);
    if (e != cudaSuccess) return e;
    if (S->p.split == VOG_SPLIT_XVX) {
        e = f64_x(S, f, f, 0.5 * dt);
        if (e == cudaSuccess) e = f64_field(S, f, nullptr);
        if (e == cudaSuccess) e = f64_v_total(S, f, S->g, dt, Eext);
        if (e == cudaSuccess) e = f64_x(S, S->g, f, 0.5 * dt);
        S->E_valid = true; S->E_of = f;        // (x-advection changes rho: E is the field solved INSIDE the step)
    } else {
        if (!(S->E_valid && S->E_of == f)) e = f64_field(S, f, nullptr);
        if (e == cudaSuccess) e = f64_v_total(S, f, S->g, 0.5 * dt, Eext);
        if (e == cudaSuccess) e = f64_x(S, S->g, S->g, dt);
        if (e == cudaSuccess) e = f64_field(S, S->g, nullptr);
        if (e == cudaSuccess) e = f64_v_total(S, S->g, f, 0.5 * dt, Eext);
        S->E_valid = true; S->E_of = f;        // (a v-advection leaves rho, hence E, unchanged: P:83)
    }
    return e;
}

}  // namespace vog
