// vog_lib.cu -- C ABI of libvog (include/vog.h): plan, shift-setup kernel (S1), density (S8) and
// Poisson (S9) kernels, and the Strang driver (S10).  The fused advection kernels (S2-S7) live in
// vog_advect.cuh.  Product code: no CPU fallback, nothing shared with oracle/.
#include <cmath>
#include <cstdio>
#include <cstdlib>
#include <cstring>
#include <new>
#include <vector>

#include "../../include/vog.h"
#include "vog_fft.cuh"
#include "vog_internal.h"

namespace vog {

// (working builds only, -DVOG_STAMPS: globaltimer stamps of the field kernels' phases)
#ifdef VOG_STAMPS
__device__ long long vog_stamps[32];
#define VOG_STAMP(i) do { if (threadIdx.x == 0) { long long t_; asm volatile("mov.u64 %0, %%globaltimer;" : "=l"(t_)); vog_stamps[i] = t_; } } while (0)
#else
#define VOG_STAMP(i) do { } while (0)
#endif

// Programmatic dependent launch is a per-plan choice (vog_plan_tune(26, .)); the entry points of the C ABI set it
// for the calling thread before they launch anything.
static thread_local bool t_pdl = true;
bool pdl_enabled()
{
    static const bool on = [] { const char* e = std::getenv("VOG_NO_PDL"); return !(e && e[0] == '1'); }();
    return on && t_pdl;
}

advect_launch_fn advect_launcher(int N)
{
    switch (N) {
        case 64: return advect_launch_64;
        case 128: return advect_launch_128;
        case 256: return advect_launch_256;
        case 512: return advect_launch_512;
    }
    return nullptr;
}

advect_x_launch_fn advect_x_launcher(int N)
{
    switch (N) {
        case 64: return advect_x_launch_64;
        case 128: return advect_x_launch_128;
        case 256: return advect_x_launch_256;
        case 512: return advect_x_launch_512;
    }
    return nullptr;
}

int advect_x_occupancy(int N, int sym, int threads, size_t smem)
{
    switch (N) {
        case 64: return advect_x_occ_64(sym, threads, smem);
        case 128: return advect_x_occ_128(sym, threads, smem);
        case 256: return advect_x_occ_256(sym, threads, smem);
        case 512: return advect_x_occ_512(sym, threads, smem);
    }
    return 0;
}

size_t advect_x_smem_bytes(int N, int lpi_log, int nbuf)
{
    return ((size_t)nbuf << lpi_log) * ((size_t)N * sizeof(float) + XREC_WORDS * sizeof(float));
}

size_t advect_smem_bytes(int N, int lognl)
{
    const size_t NL = (size_t)1 << lognl;
    return NL * padded_len(N) * sizeof(float2) + 2 * NL * REC_WORDS * sizeof(float);
}

// ------------------------------------------------------------------------------------------
// S1: per-line shift records.  beta = -c dt / Delta in fp64; b = floor(beta), b* = beta - b.
struct SetupArgs {
    int n_lines, N, mode;      // mode 0: c = v_l (x-advection); 1: c = E_l (+E_ext_l); 2: explicit beta
    int spline, d;             // interpolation: spline3 or Lagrange degree 2d+1
    double dt, delta, vmin, dv;
    const float* E;
    const float* Eext;
    const double* beta;
    float* rec;
};

__global__ void shift_setup_kernel(const SetupArgs s)
{
    const int l = blockIdx.x * blockDim.x + threadIdx.x;
    pdl_wait();                                   // E comes from the Poisson kernel; the records may still be read
    pdl_launch_dependents();
    if (l >= s.n_lines) return;
    double beta;
    float sshift = 0.0f;
    if (s.mode == 0) {
        const double v = s.vmin + (double)l * s.dv;
        beta = -v * s.dt / s.delta;
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
    double bm = fmod(fl, (double)s.N);
    if (bm < 0.0) bm += (double)s.N;
    int b = (int)bm;
    if (b >= s.N) b = 0;
    float* r = s.rec + (size_t)l * REC_WORDS;
    const double sc = 1.0 / (2.0 * (double)s.N);
    r[0] = __int_as_float(b);
    if (s.spline) {
        // cardinal cubic B-spline at b*+1, b*, b*-1, b*-2 (= B_0^3(x_{j+b*}), j = 3..0), times 3/(2N)
        const double u = 1.0 - t;
        r[1] = (float)(3.0 * sc * (u * u * u / 6.0));
        r[2] = (float)(3.0 * sc * ((4.0 - 6.0 * t * t + 3.0 * t * t * t) / 6.0));
        r[3] = (float)(3.0 * sc * ((1.0 + 3.0 * t + 3.0 * t * t - 3.0 * t * t * t) / 6.0));
        r[4] = (float)(3.0 * sc * (t * t * t / 6.0));
        for (int k = 5; k < 19; ++k) r[k] = 0.0f;
    } else {
        // a_k(t) = (-1)^k C(t+k, 2k+1): a_0 = t, a_k = a_{k-1} (k^2 - t^2) / (2k (2k+1))
        for (int half = 0; half < 2; ++half) {
            const double tt = half == 0 ? 1.0 - t : t;
            double a = tt;
            float* o = r + 1 + 9 * half;
            o[0] = (float)(a * sc);
            for (int k = 1; k <= 8; ++k) {
                a = (k <= s.d) ? a * ((double)(k * k) - tt * tt) / (double)(2 * k * (2 * k + 1)) : 0.0;
                o[k] = (float)(a * sc);
            }
        }
    }
    r[19] = sshift;
}

// S1 for the contiguous-line kernel: records of XREC_WORDS floats (layout in vog_internal.h).
__global__ void shift_setup_x_kernel(const SetupArgs s)
{
    const int l = blockIdx.x * blockDim.x + threadIdx.x;
    pdl_wait();
    pdl_launch_dependents();
    if (l >= s.n_lines) return;
    double beta;
    if (s.mode == 0) beta = -(s.vmin + (double)l * s.dv) * s.dt / s.delta;
    else beta = s.beta[l];
    const double fl = floor(beta);
    const double t = beta - fl;
    double bm = fmod(fl, (double)s.N);
    if (bm < 0.0) bm += (double)s.N;
    int b = (int)bm;
    if (b >= s.N) b = 0;
    float* r = s.rec + (size_t)l * XREC_WORDS;
    const double sc = 1.0 / (2.0 * (double)s.N);
    const double sgn = (b & 1) ? -1.0 : 1.0;
    for (int k = 0; k < XREC_WORDS; ++k) r[k] = 0.0f;
    r[0] = __int_as_float(b);
    r[1] = (float)(1.0 / (double)s.N);
    double nyq;
    if (s.spline) {
        const double u = 1.0 - t;
        const double Bm1 = u * u * u / 6.0, B0 = (4.0 - 6.0 * t * t + 3.0 * t * t * t) / 6.0;
        const double B1 = (1.0 + 3.0 * t + 3.0 * t * t - 3.0 * t * t * t) / 6.0, B2 = t * t * t / 6.0;
        r[4] = (float)(3.0 * sc * Bm1); r[5] = (float)(3.0 * sc * B0);
        r[6] = (float)(3.0 * sc * B1);  r[7] = (float)(3.0 * sc * B2);
        nyq = 3.0 * (B0 + B2 - Bm1 - B1);           // theta = pi: c = -1, s = 0, 3/(2+c) = 3
    } else {
        double p[2];
        for (int half = 0; half < 2; ++half) {
            const double tt = half == 0 ? 1.0 - t : t;
            double a = tt, pw = 1.0, acc = 0.0;
            float* o = r + 4 + 9 * half;
            for (int k = 0; k <= 8; ++k) {
                if (k > 0) a = (k <= s.d) ? a * ((double)(k * k) - tt * tt) / (double)(2 * k * (2 * k + 1)) : 0.0;
                o[k] = (float)(a * sc);
                acc += a * pw;
                pw *= 4.0;                           // s = 2 - 2 cos(pi) = 4
            }
            p[half] = acc;
        }
        nyq = p[0] - p[1];                           // P(4;1-b*) + e^{i pi} P(4;b*)
    }
    r[2] = (float)(sgn * nyq / (double)s.N);
}

// ------------------------------------------------------------------------------------------
// S8: rho partial sums.  grid (Nx/32, NBY), 256 threads: a warp covers 4 rows x 32 columns
// (8 lanes x float4 = one 128 B line per row); the 4 row-lanes are folded by warp shuffles,
// the 8 warps through shared memory; fp64 accumulation, fixed order => deterministic.  Block (x, y) writes the sums
// of its row slab to part[y][32 x .. 32 x + 31]; the Poisson kernel adds the NBY slabs in index order (no atomics,
// no "last block" pass: the slabs are <= 16 rows of Nx doubles, a few KB for the single CTA that needs them).
// KIN: also the column sums weighted with v_j^2 (kinetic energy) into partk, same layout.
template <bool KIN>
__global__ void __launch_bounds__(256) density_partial_kernel(const float* __restrict__ f, int Nx, int Nv,
                                                              int rows_per_block, double* __restrict__ part,
                                                              double* __restrict__ partk, double vmin, double dvd,
                                                              unsigned* __restrict__ tick, double* __restrict__ rho_out,
                                                              double rho_scale)
{
    __shared__ double red[8][32];
    __shared__ unsigned last_s;
    __shared__ double redk[KIN ? 8 : 1][32];
    const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
    const int xl = lane & 7, rl = lane >> 3;
    const int col = blockIdx.x * 32 + xl * 4;
    const int j0 = blockIdx.y * rows_per_block;
    pdl_wait();                                   // f comes from the advection before; part may still be read
    pdl_launch_dependents();
#ifdef VOG_STAMPS
    if (blockIdx.x == 0 && blockIdx.y == 0) VOG_STAMP(8);
#endif
    double s0 = 0, s1 = 0, s2 = 0, s3 = 0;
    double k0 = 0, k1 = 0, k2 = 0, k3 = 0;
    const float* p = f + (size_t)(j0 + warp * 4 + rl) * Nx + col;
#pragma unroll 4
    for (int j = warp * 4 + rl; j < rows_per_block; j += 32) {
        const float4 v = __ldg(reinterpret_cast<const float4*>(p));
        s0 += (double)v.x; s1 += (double)v.y; s2 += (double)v.z; s3 += (double)v.w;
        if constexpr (KIN) {
            const double vj = vmin + (double)(j0 + j) * dvd, v2 = vj * vj;
            k0 += v2 * (double)v.x; k1 += v2 * (double)v.y; k2 += v2 * (double)v.z; k3 += v2 * (double)v.w;
        }
        p += (size_t)32 * Nx;
    }
#pragma unroll
    for (int o = 8; o <= 16; o <<= 1) {
        s0 += __shfl_xor_sync(0xffffffffu, s0, o);
        s1 += __shfl_xor_sync(0xffffffffu, s1, o);
        s2 += __shfl_xor_sync(0xffffffffu, s2, o);
        s3 += __shfl_xor_sync(0xffffffffu, s3, o);
        if constexpr (KIN) {
            k0 += __shfl_xor_sync(0xffffffffu, k0, o);
            k1 += __shfl_xor_sync(0xffffffffu, k1, o);
            k2 += __shfl_xor_sync(0xffffffffu, k2, o);
            k3 += __shfl_xor_sync(0xffffffffu, k3, o);
        }
    }
    if (rl == 0) {
        red[warp][xl * 4 + 0] = s0; red[warp][xl * 4 + 1] = s1; red[warp][xl * 4 + 2] = s2; red[warp][xl * 4 + 3] = s3;
        if constexpr (KIN) { redk[warp][xl * 4 + 0] = k0; redk[warp][xl * 4 + 1] = k1; redk[warp][xl * 4 + 2] = k2; redk[warp][xl * 4 + 3] = k3; }
    }
    __syncthreads();
    if (threadIdx.x < 32) {
        double s = 0, k = 0;
#pragma unroll
        for (int w = 0; w < 8; ++w) {
            s += red[w][threadIdx.x];
            if constexpr (KIN) k += redk[w][threadIdx.x];
        }
        part[(size_t)blockIdx.y * Nx + blockIdx.x * 32 + threadIdx.x] = s;
        if constexpr (KIN) partk[(size_t)blockIdx.y * Nx + blockIdx.x * 32 + threadIdx.x] = k;
    }
    if (tick) {
        // (fused field solve, field_then_v: the v kernel's CTAs all need all of rho.)  The last block of a column group
        // to arrive adds the group's slabs in the order of poisson_kernel -- slabs 0..7, slabs 8..15, then the two
        // halves -- and writes rho_i = dv * sum: the same value whichever block comes last.
        if (threadIdx.x < 32) {
            __threadfence();
            __syncwarp();
            if (threadIdx.x == 0) last_s = atomicAdd(tick + blockIdx.x, 1u);
            __syncwarp();
            if (last_s == gridDim.y - 1u) {
                __threadfence();
                const int i = blockIdx.x * 32 + threadIdx.x, nby = (int)gridDim.y;
                double v[16];
#pragma unroll
                for (int y = 0; y < 16; ++y) v[y] = y < nby ? __ldcg(part + (size_t)y * Nx + i) : 0.0;
                double a = v[0], b = v[8];
#pragma unroll
                for (int y = 1; y < 8; ++y) { a += v[y]; b += v[8 + y]; }
                rho_out[i] = (nby > 8 ? a + b : a) * rho_scale;
                if (threadIdx.x == 0) tick[blockIdx.x] = 0u;
            }
        }
    }
#ifdef VOG_STAMPS
    if (blockIdx.x == gridDim.x - 1 && blockIdx.y == gridDim.y - 1) VOG_STAMP(9);
#endif
}

// ------------------------------------------------------------------------------------------
// NEXT-3: the paper's other field solve and its diagnostics, one CTA of 1024 threads.
//   solver 1: trapezoidal rule with the zero-mean modifications: M = mean rho, rho~ = rho - M,
//             E~_0 = 0, E~_{k+1} = E~_k + dx (rho~_k + rho~_{k+1})/2, E = E~ - mean E~;
//   solver 2: the same without them: rho~ = rho - background ("rho - 1"; minus the equilibrium's mass in
//             delta-f mode), E = E~;
//   solver 0: E is given (the Fourier solve ran before): diagnostics only.
// diag (if not NULL): [0] (1/2) dx sum E^2, [1] rho^_0 + mass0 (mass error = |.. - 1|), [2] |rho^_1|
// (P:261), [3] kinetic energy (1/2) dx dv sum_j v_j^2 sum_i f_ji + kin0, [4] total energy [0] + [3].
// All sums in fp64, fixed order.
__device__ __forceinline__ double block_sum_1024(double v, double* red, const int tid, const int T)
{
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) v += __shfl_xor_sync(0xffffffffu, v, o);
    __syncthreads();                               // red may still be read from the last call
    if ((tid & 31) == 0) red[tid >> 5] = v;
    __syncthreads();
    double s = 0.0;
    for (int w = 0; w < (T >> 5); ++w) s += red[w];
    return s;
}

__global__ void __launch_bounds__(1024) field_aux_kernel(int Nx, int solver, const double* __restrict__ part,
                                                         const double* __restrict__ partk, int nby, double dv, double dx,
                                                         double background, double mass0, double kin0,
                                                         double* __restrict__ rho, float* __restrict__ E_a,
                                                         float* __restrict__ E_b, double* __restrict__ diag)
{
    __shared__ double red[32];
    __shared__ double scan[1024];
    const int tid = threadIdx.x, T = blockDim.x;
    const int per = (Nx + T - 1) / T, i0 = tid * per, i1 = min(Nx, i0 + per);     // consecutive cells per thread
    pdl_wait();
    pdl_launch_dependents();
    // rho_i = dv * (sum of the slab sums, in slab order); K = dv sum_i (sum_j v_j^2 f_ji)
    double srho = 0.0, skin = 0.0, sre = 0.0, sim = 0.0;
    for (int i = i0; i < i1; ++i) {
        double s = 0.0;
        for (int y = 0; y < nby; ++y) s += __ldcg(part + (size_t)y * Nx + i);
        s *= dv;
        rho[i] = s;                                // (solver 0: the Fourier solve has written the same value already)
        srho += s;
        if (diag) {
            double sn, cs;
            sincospi(-2.0 * (double)i / (double)Nx, &sn, &cs);
            sre += s * cs;
            sim += s * sn;
            if (partk) {
                double k = 0.0;
                for (int y = 0; y < nby; ++y) k += __ldcg(partk + (size_t)y * Nx + i);
                skin += k;
            }
        }
    }
    const double mean = block_sum_1024(srho, red, tid, T) / (double)Nx;
    double e2 = 0.0;
    if (solver != 0) {
        __syncthreads();                           // rho[] of the neighbouring thread's first cell
        const double M = solver == 1 ? mean : background;
        // increments d_k = dx (rho~_{k-1} + rho~_k)/2 for k >= 1, d_0 = 0; E~_k = inclusive sum
        double loc = 0.0;
        for (int i = i0; i < i1; ++i)
            if (i > 0) loc += dx * ((rho[i - 1] - M) + (rho[i] - M)) * 0.5;
        scan[tid] = loc;
        __syncthreads();
        // exclusive scan of the 1024 per-thread sums (Hillis-Steele in shared memory, fp64)
        for (int o = 1; o < T; o <<= 1) {
            const double add = tid >= o ? scan[tid - o] : 0.0;
            __syncthreads();
            scan[tid] += add;
            __syncthreads();
        }
        double run = tid > 0 ? scan[tid - 1] : 0.0;
        double sE = 0.0;
        for (int i = i0; i < i1; ++i) {
            if (i > 0) run += dx * ((rho[i - 1] - M) + (rho[i] - M)) * 0.5;
            sE += run;
        }
        const double Mt = solver == 1 ? block_sum_1024(sE, red, tid, T) / (double)Nx : 0.0;
        run = tid > 0 ? scan[tid - 1] : 0.0;
        for (int i = i0; i < i1; ++i) {
            if (i > 0) run += dx * ((rho[i - 1] - M) + (rho[i] - M)) * 0.5;
            const float e = (float)(run - Mt);
            E_a[i] = e;
            if (E_b) E_b[i] = e;
            e2 += (double)e * (double)e;
        }
    } else if (diag) {
        for (int i = i0; i < i1; ++i) { const double e = (double)E_a[i]; e2 += e * e; }
    }
    if (diag) {
        const double se2 = block_sum_1024(e2, red, tid, T);
        const double re = block_sum_1024(sre, red, tid, T), im = block_sum_1024(sim, red, tid, T);
        const double kin = block_sum_1024(skin, red, tid, T);
        if (tid == 0) {
            diag[0] = 0.5 * dx * se2;
            diag[1] = mean + mass0;
            diag[2] = sqrt(re * re + im * im) / (double)Nx;
            diag[3] = 0.5 * dx * dv * kin + kin0;
            diag[4] = diag[0] + diag[3];
        }
    }
}


// S9: single-CTA Poisson solve.  rho_i = dv * sum of partials (fp64), zero mean in fp64
// (P:205-211), mixed-radix (4/8/16, in registers) DIF FFT in shared memory (fp32), E^_m = rho^_m / (i k_m)
// with modes 0 and Nx/2 dropped, DIT inverse, E written to E_a (and E_b if non-NULL).
struct PoissonRadix { int np; int lr[8]; int off[8]; };   // log2 radix and twiddle-table offset of each pass

// One pass over sub-blocks of length B = 1 << lB, radix R, stride S = B / R.  tw = the pass's compact table
// [(q-1) S + t] = e^{-2 pi i t q / B}: lanes read consecutive entries (no bank conflicts).
// Twiddles are read with explicit shared-memory loads when TWS (the table is staged in shared memory for Nx <= 8192): a
// generic pointer that may be shared or global compiles to generic loads, ~4x the latency, and they sat in the
// dependency chain of every pass (measured: 0.42 us per pass of 512 butterflies).  All loads of a butterfly are
// issued before its first store.
template <bool TWS>
__device__ __forceinline__ float2 poisson_tw(const float2* tw, const int i)
{
    if constexpr (TWS) {
        float2 v;
        const unsigned a = (unsigned)__cvta_generic_to_shared(tw + i);
        asm volatile("ld.shared.v2.f32 {%0, %1}, [%2];\n" : "=f"(v.x), "=f"(v.y) : "r"(a));
        return v;
    } else {
        return __ldg(tw + i);
    }
}

template <int R, bool INV, bool TWS>
__device__ __forceinline__ void poisson_pass(float2* __restrict__ z, const int Nx, const int lB,
                                             const float2* __restrict__ tw, const int tid, const int T,
                                             const float* __restrict__ iks)
{
    // (positions are padded by one float2 per 16, padp(): the last forward / first inverse pass has a stride of R
    // positions between neighbouring threads, which would put a warp on few bank pairs)
    constexpr int LR = ilog2(R);
    const int lS = lB - LR, S = 1 << lS;
#pragma unroll 1
    for (int g = tid; g < (Nx >> LR); g += T) {
        const int t = g & (S - 1), base = ((g >> lS) << lB) + t;
        float2 x[R], w[R];
#pragma unroll
        for (int q = 1; q < R; ++q) w[q] = poisson_tw<TWS>(tw, ((q - 1) << lS) + t);
        if constexpr (!INV) {
#pragma unroll
            for (int k = 0; k < R; ++k) x[k] = z[padp(base + (k << lS))];
            dft_dif<R, 1>(x);
            z[padp(base)] = x[0];
#pragma unroll
            for (int q = 1; q < R; ++q) z[padp(base + (q << lS))] = cmul(x[brev(q, R)], w[q]);
        } else {
            // iks != NULL (first inverse pass): the spectrum is divided by i k on the way in, (zr + i zi) / (i k) / Nx
            float2 v[R];
#pragma unroll
            for (int q = 0; q < R; ++q) v[q] = z[padp(base + (q << lS))];
            if (iks) {
#pragma unroll
                for (int q = 0; q < R; ++q) {
                    const float ik = iks[base + (q << lS)];
                    v[q] = make_float2(v[q].y * ik, -v[q].x * ik);
                }
            }
            x[0] = v[0];
#pragma unroll
            for (int q = 1; q < R; ++q) x[brev(q, R)] = cmulc(v[q], w[q]);
            idft_dit<R, 1>(x);
#pragma unroll
            for (int k = 0; k < R; ++k) z[padp(base + (k << lS))] = x[k];
        }
    }
}

// forward passes, then the inverse passes in reverse order (the first inverse pass divides by i k); ONE radix-4 body
// per direction in a run-time loop, plus one radix-2 pass when log2 Nx is odd.  Twiddle tables follow one another in
// pass order: radix R at block size B takes (R - 1) B / R entries.
template <bool INV, bool TWS>
__device__ __forceinline__ void poisson_pass_r(const int lr, float2* __restrict__ z, const int Nx, const int lB,
                                               const float2* __restrict__ tw, const int tid, const int T,
                                               const float* __restrict__ iks)
{
    if (lr == 1) poisson_pass<2, INV, TWS>(z, Nx, lB, tw, tid, T, iks);
    else if (lr == 2) poisson_pass<4, INV, TWS>(z, Nx, lB, tw, tid, T, iks);
    else poisson_pass<8, INV, TWS>(z, Nx, lB, tw, tid, T, iks);
}

// forward passes, then the inverse passes in reverse order (the first inverse pass divides by i k).  Radix 2^LR passes
// in a run-time loop (one body per direction), preceded by one pass of radix 2^(log2 Nx mod LR) when LR does not divide
// log2 Nx.  Twiddle tables follow one another in pass order: radix R at block size B takes (R - 1) B / R entries.
template <bool TWS, int LR>
__device__ __forceinline__ void poisson_fft(float2* __restrict__ z, const int Nx, const float2* __restrict__ tws,
                                            const float* __restrict__ iks, const int tid, const int T)
{
    constexpr int R = 1 << LR;
    const int lg = ilog2(Nx), rem = lg % LR;
    int lB = lg;
    const float2* tw = tws;
    if (rem) {
        poisson_pass_r<false, TWS>(rem, z, Nx, lB, tw, tid, T, nullptr);
        tw += ((1 << rem) - 1) << (lB - rem);
        lB -= rem;
        __syncthreads();
    }
#pragma unroll 1
    for (; lB > 0; lB -= LR) {
        poisson_pass<R, false, TWS>(z, Nx, lB, tw, tid, T, nullptr);
        tw += (R - 1) << (lB - LR);
        __syncthreads();
    }
    VOG_STAMP(4);
#pragma unroll 1
    for (lB = LR; lB <= lg - rem; lB += LR) {
        tw -= (R - 1) << (lB - LR);
        poisson_pass<R, true, TWS>(z, Nx, lB, tw, tid, T, lB == LR ? iks : nullptr);
        __syncthreads();
    }
    if (rem) {
        poisson_pass_r<true, TWS>(rem, z, Nx, lg, tws, tid, T, nullptr);
        __syncthreads();
    }
}

// S9: single-CTA Poisson solve.  rho (fp64, the density kernel's slab sums added in slab order) minus a
// reference value in fp64 (zero mean, = mode 0 dropped); DIF FFT in shared memory (fp32) in at most four
// register-resident passes -- radix 16, preceded by one radix 2, 4 or 8 pass when log2 Nx is not a multiple of 4:
// 2048 = 8 x 16 x 16 (a single SM runs this kernel, so its time is the number of barrier-separated passes: three
// fat ones instead of the five thin radix-4 ones of round 1); E^_m = rho^_m / (i k_m) with modes 0 and Nx/2
// dropped, applied while the first inverse pass loads; DIT inverse; E to E_a (and E_b).
__global__ void __launch_bounds__(1024) poisson_kernel(int Nx, const PoissonRadix rx, int tw_len, int tw_in_smem,
                                                       const float2* __restrict__ tw_g, const float* __restrict__ ikt,
                                                       const double* __restrict__ part, int nby, double dv,
                                                       double* __restrict__ rho, float* __restrict__ E_a,
                                                       float* __restrict__ E_b, double* __restrict__ energy_out,
                                                       double half_dx)
{
    __shared__ double ered[32];
    extern __shared__ __align__(16) unsigned char smem_raw[];
    float2* z = reinterpret_cast<float2*>(smem_raw);
    float* iks = reinterpret_cast<float*>(z + padded_len(Nx));      // 1/(i k) factors
    float2* twsm = reinterpret_cast<float2*>(iks + Nx); // compact twiddle tables of all passes (if they fit)
    const int tid = threadIdx.x, T = blockDim.x;
    // Zero mean = mode 0 dropped below.  Before the conversion to fp32 a constant of the size of
    // the mean must still be removed in fp64 (in full-f mode rho ~ 1 carries a 1e-3 perturbation): rho[0]
    // serves as well as the mean (any constant only changes mode 0) and needs no reduction.
    VOG_STAMP(0);
    for (int i = tid; i < Nx; i += T) iks[i] = __ldg(ikt + i);               // (plan constants: before the wait)
    if (tw_in_smem)
        for (int i = tid; i < tw_len; i += T) twsm[i] = __ldg(tw_g + i);
    pdl_wait();                                   // the slab sums come from the density kernel
    pdl_launch_dependents();
    // rho_i = dv * (sum of the slab sums, in slab order); rho_0 is the reference value
    // rho_i = dv * (sum of the slab sums in a fixed order: slabs 0..7, then slabs 8..15, then the two halves).  The eight
    // values of a half are requested before the first is used, and the reference cell 0 travels with the thread's
    // first cell: one L2 round trip for the first 1024 cells, one more per further 1024.
    auto slab8 = [&](const int i, const int y0) {
        double v[8];
#pragma unroll
        for (int y = 0; y < 8; ++y) v[y] = y0 + y < nby ? __ldcg(part + (size_t)(y0 + y) * Nx + i) : 0.0;
        double s = v[0];
#pragma unroll
        for (int y = 1; y < 8; ++y) s += v[y];
        return s;
    };
    const double ref0 = slab8(0, 0);
    double s_first = slab8(tid, 0);                // (T <= Nx)
    double ref = ref0;
    if (nby > 8) { ref += slab8(0, 8); s_first += slab8(tid, 8); }
    ref *= dv;
    s_first *= dv;
    rho[tid] = s_first;
    z[padp(tid)] = make_float2((float)(s_first - ref), 0.0f);
#pragma unroll 1
    for (int i = tid + T; i < Nx; i += T) {
        double sv = slab8(i, 0);
        if (nby > 8) sv += slab8(i, 8);
        sv *= dv;
        rho[i] = sv;
        z[padp(i)] = make_float2((float)(sv - ref), 0.0f);
    }
    __syncthreads();
    VOG_STAMP(3);
    // forward, decimation in frequency: position ((q0 r1 + q1) r2 + q2).. holds mode q0 + r0 (q1 + r1 (q2 + ..));
    // ikt[pos] = L / (2 pi m Nx) for that mode (0 for modes 0 and Nx/2)
    if (tw_in_smem) poisson_fft<true, 3>(z, Nx, twsm, iks, tid, T);
    else poisson_fft<false, 3>(z, Nx, tw_g, iks, tid, T);
    VOG_STAMP(5);
    double e2 = 0.0;
    for (int i = tid; i < Nx; i += T) {
        const float e = z[padp(i)].x;
        E_a[i] = e;
        if (E_b) E_b[i] = e;
        e2 += (double)e * (double)e;
    }
    if (energy_out) {   // electric energy (1/2) dx sum_i E_i^2, fp64, fixed summation order
#pragma unroll
        for (int o = 16; o > 0; o >>= 1) e2 += __shfl_xor_sync(0xffffffffu, e2, o);
        if ((tid & 31) == 0) ered[tid >> 5] = e2;
        __syncthreads();
        if (tid == 0) {
            double s = 0.0;
            for (int w = 0; w < (T >> 5); ++w) s += ered[w];
            energy_out[0] = half_dx * s;
        }
    }
    VOG_STAMP(6);
}

// ------------------------------------------------------------------------------------------
// S9 in x space (steps on grids of 4096 columns or more; the 2048-column grids do the same inside the v kernel, see
// osv7_kernel).  The Fourier solve of P:221 is a circular convolution, E_i = sum_j G_{i-j} rho_j, with the Green's function
// G_n = (1/Nx) sum_{m != 0, Nx/2} e^{2 pi i m n / Nx} / (i k_m), k_m = 2 pi m / L (a plan constant, computed on the host
// in fp64: green_host).  One CTA of 1024 threads per 64 columns instead of ONE CTA for the whole solve (poisson_kernel
// takes 20 us at Nx = 8192: a single SM, ten barrier-separated passes): thread = (8 columns, a chunk of Nx / 128
// consecutive cells j) with a rolling window of G in registers -- one value of rho, one new value of G and eight
// multiply-adds per cell, fp32 (<= 128 products per partial sum); the partial sums meet in fp64 in a fixed order.
// rho comes from the density kernel's last blocks (ticket), minus rho_0, rounded to fp32 like poisson_kernel's input.
__global__ void __launch_bounds__(1024) green_field_kernel(int Nx, const double* __restrict__ green,
                                                           const double* __restrict__ rho, float* __restrict__ E_a,
                                                           double* __restrict__ energy_out, double* __restrict__ e_part,
                                                           unsigned* __restrict__ ticket, double half_dx)
{
    extern __shared__ __align__(16) unsigned char smem_raw[];
    __shared__ double eS[8];
    // G padded by one word per 8 (index x + (x >> 3)): the 32 lanes of a warp -- 8 octets of columns x 4 chunks -- read
    // G at distances 8 oct - JC jp, which this padding spreads over 32 different banks at Nx = 4096 and 8192 (two
    // wavefronts remain at 16384); rho chunk by chunk with one word between chunks (chunk jp at jp (JC + 1)).
    const int JC = Nx >> 7, PG = Nx + (Nx >> 3), PR = Nx + 128;
    float* const gS = reinterpret_cast<float*>(smem_raw);
    float* const rS = gS + PG;
    double* const sumS = reinterpret_cast<double*>(rS + PR);              // [32 warps][64 columns]
    const int tid = threadIdx.x, xmask = Nx - 1;
    for (int i = tid; i < Nx; i += 1024) gS[i + (i >> 3)] = (float)__ldg(green + i);      // (plan constant: before the wait)
    if (blockIdx.x == 0) VOG_STAMP(10);
    pdl_wait();                                   // rho comes from the density kernel
    pdl_launch_dependents();
    if (blockIdx.x == 0) VOG_STAMP(11);
    const double ref = __ldcg(rho);
    const int jsh = 31 - __clz(JC);
    for (int i = tid; i < Nx; i += 1024) rS[i + (i >> jsh)] = (float)(__ldcg(rho + i) - ref);
    __syncthreads();
    if (blockIdx.x == 0) VOG_STAMP(12);
    const int oct = tid & 7, jp = tid >> 3, j0 = jp * JC;
    const int gb = (int)blockIdx.x * 64 + 8 * oct + 7 - j0;               // index of G for column c0 + 7 at cell j0
    const float* const rp = rS + jp * (JC + 1);
    float w[8], acc[8];
#pragma unroll
    for (int k = 0; k < 8; ++k) acc[k] = 0.0f;                             // acc[k]: column 64 blockIdx.x + 8 oct + 7 - k
#pragma unroll
    for (int k = 0; k < 7; ++k) { const int gi = (gb - k) & xmask; w[k] = gS[gi + (gi >> 3)]; }
    // cells in groups of eight: G indices gb - 7 - i run from a multiple of 8 downwards, so the first lies in one padded
    // group of 8 and the other seven, contiguous, in the group below: two address computations per 8 cells
#pragma unroll 1
    for (int i0 = 0; i0 < JC; i0 += 8) {
        const int g0 = (gb - 7 - i0) & xmask, g1 = (g0 - 1) & xmask;
        const float* const q1 = gS + g1 + (g1 >> 3);
        float gv[8];
        gv[0] = gS[g0 + (g0 >> 3)];
#pragma unroll
        for (int m = 1; m < 8; ++m) gv[m] = q1[1 - m];
#pragma unroll
        for (int m = 0; m < 8; ++m) {
            w[7] = gv[m];
            const float rj = rp[i0 + m];
#pragma unroll
            for (int k = 0; k < 8; ++k) acc[k] = fmaf(w[k], rj, acc[k]);
#pragma unroll
            for (int k = 0; k < 7; ++k) w[k] = w[k + 1];
        }
    }
    if (blockIdx.x == 0) VOG_STAMP(13);
    // the four chunks of a warp by shuffles, the 32 warps through shared memory
#pragma unroll
    for (int k = 0; k < 8; ++k) {
        double d = (double)acc[k];
        d += __shfl_xor_sync(0xffffffffu, d, 8);
        d += __shfl_xor_sync(0xffffffffu, d, 16);
        if ((tid & 31) < 8) sumS[(tid >> 5) * 64 + 8 * oct + 7 - k] = d;
    }
    __syncthreads();
    if (blockIdx.x == 0) VOG_STAMP(14);
    double e2 = 0.0;
    if (tid < 256) {
        const int col = tid >> 2, part = tid & 3;
        double sv = 0.0;
#pragma unroll
        for (int q = 0; q < 8; ++q) sv += sumS[(8 * part + q) * 64 + col];
        sv += __shfl_xor_sync(0xffffffffu, sv, 1);
        sv += __shfl_xor_sync(0xffffffffu, sv, 2);
        if (part == 0) {
            const float ef = (float)sv;
            E_a[blockIdx.x * 64 + col] = ef;
            e2 = (double)ef * (double)ef;
        }
    }
    if (blockIdx.x == 0) VOG_STAMP(15);
    if (energy_out) {   // (1/2) dx sum_i E_i^2: CTA sums in CTA order by the last CTA to arrive
        if (tid < 256) {
#pragma unroll
            for (int o = 16; o > 0; o >>= 1) e2 += __shfl_xor_sync(0xffffffffu, e2, o);
            if ((tid & 31) == 0) eS[tid >> 5] = e2;
        }
        __syncthreads();
        if (tid == 0) {
            double tot = 0.0;
            for (int q = 0; q < 8; ++q) tot += eS[q];
            e_part[blockIdx.x] = tot;
            __threadfence();
            if (atomicAdd(ticket, 1u) == gridDim.x - 1u) {
                __threadfence();
                tot = 0.0;
                for (int q = 0; q < (int)gridDim.x; ++q) tot += __ldcg(e_part + q);
                energy_out[0] = half_dx * tot;
                *ticket = 0u;
            }
        }
    }
}

}  // namespace vog

// ==========================================================================================
struct vog_plan_s {
    vog_params_t p;
    cudaStream_t st;
    int sym, d;                 // symbol variant and Lagrange half-width
    float2 *tw_x, *tw_v;        // roots of unity of order Nx / Nv
    float2 *xtwA, *xtwB, *xcs;  // x kernel: pass-A twiddles [R1-1][S1], pass-B twiddles [15][16], (cos,sin)(2 pi k/Nx)
    float* xrec;                // x kernel shift records [Nv][XREC_WORDS]
    int x_nbuf;
    // overlap-save path (line length >= 1024)
    bool os_x, os_v;
    float2 *os_lam_x, *os_lam_v;   // symbol tables [Nv][OS_LAMW], [Nx][OS_LAMW]
    float2* os_twv;                // [15][16] e^{-2 pi i t q / 256}
    double2* os_cs64;
    float* cg4;                    // f_eq exponents c_g as floats
    float* ikt;                    // Poisson: 1/(i k) factor per digit-reversed position
    float2* ptw;                   // Poisson: compact per-pass twiddle tables
    int ptw_len;
    vog::PoissonRadix prx;
    float* g_buf;                  // second grid for the out-of-place v kernel (allocated on first use)
    int os2x_lpi, os3x_occ, os2v_gpc;      // x: lines per iteration, cached occupancy; v: pairs per CTA (0 = default)
    vog::OsSetupArgs vsetup;               // v-advection: shift source (E, E_ext, beta, dt) of the pending advection
    int small_run;                         // vog_run on grids up to 256 x 256 as one persistent kernel (vog_small.cu): 0 / 1
    int solver;                            // field solve: 0 = Fourier (default), 1 = trapezoid + zero mean, 2 = trapezoid, rho - 1
    double feq_mass, feq_kin;              // dv sum_j f_eq(v_j) and (1/2) L dv sum_j v_j^2 f_eq(v_j) (0 in full-f mode)
    double *partk, *diag;                  // kinetic-energy slab sums [nby_max][Nx]; 5 doubles of scratch
    int method;                            // advection of lines >= 1024 cells: 0 = in Fourier space (default, the graded path), 1 = direct stencil (NEXT-4)
    float *taps_x, *taps_v;                // stencil path: taps [Nv][32] and, transposed, [32][Nx + 16]
    int stx_occ;
    int osv_variant;                       // v kernel: 0 = 16-column strips, next window in flight (osv6_kernel, default), 1 = 32-column strips (osv4_kernel)
    int osx_variant;                       // x kernel: 0 = per-pair windows when a group fits one round (osx7_kernel), else whole lines; 1 = whole lines always (osx6_kernel)
    int pdl;                               // programmatic dependent launch of the step's kernels (default: grids up to 8192^2)
    int os_geom;                           // block geometry: 1 = Lagrange (232 kept, 8 + 16 discarded), 0 = spline (224, 16 + 16)
    int x_lpi_log, x_thr, x_cps, x_occ;   // lines per iteration (log2), threads, CTAs per SM (0 = occupancy), cached occupancy
    float *rec_x, *rec_v;       // shift records: [Nv] for x-lines, [Nx] for v-lines
    double* part;               // density partials [nby][Nx]
    double* rho;                // [Nx]
    float* E_self;              // [Nx] last self-consistent field
    double* green;              // [Nx] Green's function of the Fourier solve (plans whose v kernel can solve the field itself)
    double* e_part;             // [Nx / 16] + ticket word: energy reduction of the fused field solve
    int fuse_field;             // steps: density -> v kernel with the field solve inside (no Poisson launch); 0 / 1
    int v_spec;                 // v kernel: first windows requested before the shifts are known (default 1)
    int v_inplace;              // vog_advect_v / vog_shift_v: the v kernel stores in place where the shifts allow it (default 1)
    int* strip_flags;           // [Nx / 16] strips of the last in-place v-advection that went to the second grid
    float* ip_halo;             // [n_sm][4][2][40][16] boundary rows of the in-place v kernel's pieces
    int density_pdl;            // density kernel launched with the programmatic-dependent-launch attribute (0 / 1)
    bool v_behind_field;        // ... set by field_then_v around its v launch
    bool v_inplace_now;         // set by advect_v_inplace around its v launch
    float *feq_tab, *vmu_tab;   // [ng][Nv]
    int nby, nby_max;           // density: row slabs per column group (tunable up to the allocated nby_max)
    int lognl_x, lognl_v, thr_x, thr_v;
    int n_sm;
    bool E_valid;               // E_self holds a field (vog_get_field)
    const float* E_of;          // ... and it is the self-consistent field of the state in this array as the last
                                // call on the plan left it (VXV steps may then skip their first field solve); NULL otherwise
    bool recx_valid; double recx_dt;
    long long launches;
    vog::F64State* f64;         // double-precision mode (NEXT-2), created on the first *_f64 call
    float* f_buf;               // only for vog_run_host
    float* ext_buf;
};

using namespace vog;

static int ilog2i(int n) { int l = 0; while ((1 << l) < n) ++l; return l; }

// Green's function of the Fourier field solve on the host: G_n = (1/N) sum_{m != 0, N/2} e^{2 pi i m n / N} / (i k_m),
// k_m = 2 pi m / L with m counted from -N/2: the inverse transform of the solver's own factors, by a plain radix-2
// transform in fp64 (N <= 16384 is a power of two).  Real by symmetry.
static void green_host(int N, double L, std::vector<double>& G)
{
    const long double PI = 3.14159265358979323846264338327950288L;
    std::vector<double> re(N, 0.0), im(N, 0.0);
    for (int m = 1; m < N; ++m) {
        if (2 * m == N) continue;
        const int ms = m < N / 2 ? m : m - N;
        im[m] = (double)(-(long double)L / (2.0L * PI * (long double)ms * (long double)N));      // 1 / (i k) = -i / k
    }
    const int lg = ilog2i(N);
    for (int i = 0; i < N; ++i) {                  // bit reversal
        int r = 0;
        for (int b = 0; b < lg; ++b) r |= ((i >> b) & 1) << (lg - 1 - b);
        if (r > i) { std::swap(re[i], re[r]); std::swap(im[i], im[r]); }
    }
    for (int len = 2; len <= N; len <<= 1) {       // decimation in time, e^{+2 pi i / len}
        const int half = len / 2;
        std::vector<double> wr(half), wi(half);
        for (int k = 0; k < half; ++k) {
            const long double a = 2.0L * PI * (long double)k / (long double)len;
            wr[k] = (double)cosl(a); wi[k] = (double)sinl(a);
        }
        for (int i0 = 0; i0 < N; i0 += len)
            for (int k = 0; k < half; ++k) {
                const int p = i0 + k, q = p + half;
                const double tr = re[q] * wr[k] - im[q] * wi[k], ti = re[q] * wi[k] + im[q] * wr[k];
                re[q] = re[p] - tr; im[q] = im[p] - ti;
                re[p] += tr; im[p] += ti;
            }
    }
    G.assign(re.begin(), re.end());
}
static bool pow2_in_range(int n) { return n >= 64 && n <= 16384 && (n & (n - 1)) == 0; }

static void fill_roots(std::vector<float2>& h, int N)
{
    h.resize(N);
    for (int k = 0; k < N; ++k) {
        // e^{-2 pi i k / N}, exact on the axes, long double elsewhere, rounded once
        float c, s;
        if ((4 * k) % N == 0) {
            const int q = (4 * k) / N;
            c = q == 0 ? 1.f : (q == 2 ? -1.f : 0.f);
            s = q == 1 ? 1.f : (q == 3 ? -1.f : 0.f);
        } else {
            const long double a = 2.0L * 3.14159265358979323846264338327950288L * (long double)k / (long double)N;
            c = (float)cosl(a);
            s = (float)sinl(a);
        }
        h[k] = make_float2(c, -s);
    }
}

// e^{-2 pi i k / n}, exact on the axes and diagonals' signs, long double elsewhere, rounded once
static float2 unit_root_neg(long long k, long long n)
{
    k %= n;
    if (k < 0) k += n;
    if ((4 * k) % n == 0) {
        const int q = (int)((4 * k) / n);
        return make_float2(q == 0 ? 1.f : (q == 2 ? -1.f : 0.f), q == 1 ? -1.f : (q == 3 ? 1.f : 0.f));
    }
    const long double a = 2.0L * 3.14159265358979323846264338327950288L * (long double)k / (long double)n;
    return make_float2((float)cosl(a), -(float)sinl(a));
}

static void x_radix(int N, int* R1, int* R2)
{
    switch (N) {
        case 64: *R1 = 2; *R2 = 1; break;
        case 128: *R1 = 4; *R2 = 1; break;
        case 256: *R1 = 8; *R2 = 1; break;
        case 512: *R1 = 16; *R2 = 1; break;
        case 1024: *R1 = 32; *R2 = 1; break;
        case 2048: *R1 = 4; *R2 = 16; break;
        case 4096: *R1 = 8; *R2 = 16; break;
        case 8192: *R1 = 16; *R2 = 16; break;
        default: *R1 = 32; *R2 = 16; break;
    }
}

// twiddle tables of the contiguous-line kernel for line length N (complex length M = N/2)
static void fill_x_tables(int N, std::vector<float2>& twA, std::vector<float2>& twB, std::vector<float2>& cs)
{
    int R1, R2;
    x_radix(N, &R1, &R2);
    const int M = N / 2, S1 = M / R1;
    twA.assign((size_t)(R1 - 1) * S1, make_float2(1.f, 0.f));
    for (int q = 1; q < R1; ++q)
        for (int t = 0; t < S1; ++t) twA[(size_t)(q - 1) * S1 + t] = unit_root_neg((long long)t * q, M);
    twB.assign(15 * 16, make_float2(1.f, 0.f));
    for (int q = 1; q < 16; ++q)
        for (int t = 0; t < 16; ++t) twB[(q - 1) * 16 + t] = unit_root_neg(t * q, 256);
    cs.resize(M + 1);
    for (int k = 0; k <= M; ++k) {
        const float2 w = unit_root_neg(k, N);
        cs[k] = make_float2(w.x, -w.y);          // (cos, sin)(2 pi k / N)
    }
}

static void default_x_tile(int N, int n_lines, int* lpi_log, int* threads)
{
    int lpi = 8192 / N;
    if (lpi < 1) lpi = 1;
    if (lpi > 16) lpi = 16;
    while (lpi > 1 && n_lines / lpi < 148 * 4) lpi >>= 1;
    while (lpi > n_lines) lpi >>= 1;
    int t = lpi * (N / 64);
    if (t < 32) t = 32;
    if (t > 128) t = 128;
    *lpi_log = ilog2i(lpi);
    *threads = t;
}

// default tile shape: NL complex lines per CTA and threads per CTA (kernel section)
static void default_tile(int N, int n_lines, bool vdir, int* lognl, int* threads)
{
    const int pairs = n_lines / 2;
    int nl;
    if (N >= 16384) { *lognl = 0; *threads = 512; return; }
    if (vdir) {
        nl = N <= 2048 ? 4 : (N <= 4096 ? 2 : 1);
    } else {
        nl = 8192 / N;
        if (nl < 1) nl = 1;
        if (nl > 16) nl = 16;
    }
    while (nl > 1 && pairs / nl < 592) nl >>= 1;
    if (nl > pairs) nl = pairs;
    int t = nl * (N / 32);
    if (t < 64) t = 64;
    if (t > 256) t = 256;
    *lognl = ilog2i(nl);
    *threads = t;
}

extern "C" const char* vog_strerror(int status)
{
    switch (status) {
        case VOG_OK: return "ok";
        case VOG_EINVAL: return "invalid argument";
        case VOG_ENOMEM: return "out of device memory";
        case VOG_ECUDA: return "CUDA error";
        case VOG_EUNSUPPORTED: return "unsupported interpolation kind/order";
        case VOG_ETOOLARGE: return "size beyond the fixed scratch of the allocation-free entry point (VOG_NOALLOC_MAX_NX)";
    }
    return "unknown status";
}

static void free_plan(vog_plan_s* P)
{
    if (!P) return;
    cudaFree(P->taps_x); cudaFree(P->taps_v); cudaFree(P->os_lam_x); cudaFree(P->os_lam_v); cudaFree(P->os_twv); cudaFree(P->os_cs64); cudaFree(P->ikt); cudaFree(P->ptw); cudaFree(P->cg4);
    cudaFree(P->g_buf);
    vog::f64_destroy(P->f64);
    cudaFree(P->xtwA); cudaFree(P->xtwB); cudaFree(P->xcs); cudaFree(P->xrec);
    cudaFree(P->tw_x); cudaFree(P->tw_v); cudaFree(P->rec_x); cudaFree(P->rec_v);
    cudaFree(P->part); cudaFree(P->partk); cudaFree(P->diag); cudaFree(P->rho); cudaFree(P->E_self); cudaFree(P->green); cudaFree(P->e_part); cudaFree(P->strip_flags); cudaFree(P->ip_halo);
    cudaFree(P->feq_tab); cudaFree(P->vmu_tab); cudaFree(P->f_buf); cudaFree(P->ext_buf);
    delete P;
}

extern "C" int vog_plan(vog_plan_t* out, const vog_params_t* p, void* cuda_stream)
{
    if (!out || !p) return VOG_EINVAL;
    if (!pow2_in_range(p->Nx) || !pow2_in_range(p->Nv)) return VOG_EINVAL;
    if (!(p->L > 0.0) || !(p->vmax > p->vmin) || !std::isfinite(p->L) || !std::isfinite(p->vmin) || !std::isfinite(p->vmax))
        return VOG_EINVAL;
    if (p->feq.n < 0 || p->feq.n > 4) return VOG_EINVAL;
    for (int g = 0; g < p->feq.n; ++g)
        if (!(p->feq.c[g] > 0.0) || !std::isfinite(p->feq.amp[g]) || !std::isfinite(p->feq.mu[g])) return VOG_EINVAL;
    if (p->split != VOG_SPLIT_XVX && p->split != VOG_SPLIT_VXV) return VOG_EINVAL;
    int sym, d = 0;
    const int nmin = p->Nx < p->Nv ? p->Nx : p->Nv;
    if (p->kind == VOG_LAGRANGE) {
        if (p->order < 1 || p->order > 17 || (p->order & 1) == 0 || p->order > nmin - 1) return VOG_EUNSUPPORTED;
        d = (p->order - 1) / 2;
        sym = d <= 1 ? SYM_LAG_D1 : (d <= 4 ? SYM_LAG_D4 : SYM_LAG_D8);
    } else if (p->kind == VOG_BSPLINE) {
        if (p->order != 3) return VOG_EUNSUPPORTED;
        sym = SYM_SPLINE3;
    } else {
        return VOG_EUNSUPPORTED;
    }
    vog_plan_s* P = new (std::nothrow) vog_plan_s();
    if (!P) return VOG_ENOMEM;
    std::memset(P, 0, sizeof(*P));
    P->p = *p;
    P->st = (cudaStream_t)cuda_stream;
    P->sym = sym;
    P->d = d;
    const int Nx = p->Nx, Nv = p->Nv, ng = p->feq.n;
    // density row slabs per column group: up to 512 blocks of at least 128 rows, and never more slabs than the
    // partial-sum buffer has rows (measured on 1024^2 .. 8192^2: more blocks cost more in the ticket reduction than
    // they gain in parallelism)
    P->nby_max = 16;
    int nby = 1;
    while ((Nx / 32) * nby * 2 <= 512 && Nv / (nby * 2) >= 128 && nby * 2 <= P->nby_max) nby *= 2;
    P->nby = nby;
    {
        int dev = 0, nsm = 148;
        if (cudaGetDevice(&dev) == cudaSuccess) cudaDeviceGetAttribute(&nsm, cudaDevAttrMultiProcessorCount, dev);
        P->n_sm = nsm > 0 ? nsm : 148;
    }
    default_tile(Nx, Nv, false, &P->lognl_x, &P->thr_x);
    default_x_tile(Nx, Nv, &P->x_lpi_log, &P->x_thr);
    P->os_x = Nx >= 1024;
    P->os_v = Nv >= 1024;
    P->v_spec = 1;
    P->v_inplace = 1;
    // (measured: behind an x kernel of a grid of 4096^2 cells or more the density kernel's 512 long-running blocks do
    // worse when they trickle onto the SMs as the x kernel drains -- 8192^2 step 484 us with the attribute, 451 us
    // without; on the 2048^2 grid the early start wins: 51.6 against 54.7 us)
    P->density_pdl = (long long)Nx * Nv < 4096LL * 4096LL ? 1 : 0;
    {
        // pair kernels: 16 items per pair and phase; lines per iteration so that one round of <= 320 threads
        // covers the items (8192: 18 pairs = 288 items; 2048: 3 lines x 5 pairs = 240)
        const int Vx = p->kind == VOG_LAGRANGE ? OS_VL : OS_V;
        const int npx = ((Nx + Vx - 1) / Vx + 1) / 2;
        int l2 = 288 / (16 * npx);
        if (l2 > 2) l2 = 2;                          // measured (2048, 4096 cells): 2 lines per group, then 1, then 3
        if (l2 < 1) l2 = 1;
        while (l2 > 1 && (Nv + l2 - 1) / l2 < P->n_sm * 3) --l2;
        P->os_geom = p->kind == VOG_LAGRANGE ? 1 : 0;
        P->os2x_lpi = l2; P->os3x_occ = 0; P->os2v_gpc = 0;
        // Which x kernel (measured at the end of round 2, same box, vog_plan_tune(21, .)): lines of 1024 / 2048 cells: the
        // whole-line kernel osx6_kernel -- alone as fast as the per-pair-window kernel osx7_kernel (12.3 us at 2048^2),
        // in the chain of a step 0.55 us per step faster (46.44 -> 45.85 us); 4096 cells: osx7_kernel (step 134.7
        // against 136.2 us); 8192 cells: osx6_kernel again (116.5 against 121.7 us per launch, step 432 against 441 us);
        // 16384 cells need two rounds per line, which only osx6_kernel does.
        P->osx_variant = Nx == 4096 ? 0 : 1;
    }
    // measured (profiles/r1i_pdl_setup.md): 512^2 step -20 %, 2048^2 -15 %, 8192^2 +-0; the +1.3 % at 16384^2 of round 1
    // was the density kernel (launched without the attribute on large grids since, see density_pdl): now -0.5..-4 %
    P->pdl = 1;
    P->x_nbuf = 1;   // measured: 4 single-buffered CTAs/SM beat 3 double-buffered ones (L1 keeps the twiddles)
    default_tile(Nv, Nx, true, &P->lognl_v, &P->thr_v);
    cudaError_t e = cudaSuccess;
    auto alloc = [&](void** ptr, size_t bytes) { if (e == cudaSuccess) e = cudaMalloc(ptr, bytes ? bytes : 16); };
    alloc((void**)&P->tw_x, sizeof(float2) * Nx);
    alloc((void**)&P->tw_v, sizeof(float2) * Nv);
    alloc((void**)&P->rec_x, sizeof(float) * REC_WORDS * Nv);
    alloc((void**)&P->xrec, sizeof(float) * XREC_WORDS * Nv);
    std::vector<float2> xa, xb, xc;
    fill_x_tables(Nx, xa, xb, xc);
    std::vector<float2> otv(240);
    for (int q = 1; q < 16; ++q)
        for (int t = 0; t < 16; ++t) otv[(q - 1) * 16 + t] = unit_root_neg(t * q, 256);
    alloc((void**)&P->os_twv, sizeof(float2) * otv.size());
    std::vector<double2> ocs64(OS_LB);
    for (int j = 0; j < OS_LB; ++j) {
        const int q4 = (4 * j) / OS_LB;
        if ((4 * j) % OS_LB == 0) ocs64[j] = make_double2(q4 == 0 ? 1.0 : (q4 == 2 ? -1.0 : 0.0), q4 == 1 ? 1.0 : (q4 == 3 ? -1.0 : 0.0));
        else {
            const long double a = 2.0L * 3.14159265358979323846264338327950288L * (long double)j / (long double)OS_LB;
            ocs64[j] = make_double2((double)cosl(a), (double)sinl(a));
        }
    }
    alloc((void**)&P->os_cs64, sizeof(double2) * ocs64.size());
    std::vector<float> ikt(Nx);
    std::vector<float2> ptw;
    {
        int lg = ilog2i(Nx);
        P->prx.np = 0;
        for (int i = 0; i < 8; ++i) { P->prx.lr[i] = 0; P->prx.off[i] = 0; }
        // radix 8, preceded by one radix 2 or 4 pass (measured at 2048 with the phases of the kernel time-stamped:
        // radix 4, 8 and 16 plans are within the run-to-run noise of one another once the twiddles are explicit
        // shared-memory loads; radix 8 with Nx / 4 threads was the best by a little)
        const int mr = 3;
        if (lg % mr) { P->prx.lr[P->prx.np++] = lg % mr; lg -= lg % mr; }      // the odd radix first
        while (lg > 0) { P->prx.lr[P->prx.np++] = mr; lg -= mr; }
        int Bp = Nx;
        for (int q = 0; q < P->prx.np; ++q) {             // compact twiddles [(j-1) S + t] = e^{-2 pi i t j / B}
            const int R = 1 << P->prx.lr[q], S = Bp / R;
            P->prx.off[q] = (int)ptw.size();
            for (int j = 1; j < R; ++j)
                for (int t = 0; t < S; ++t) ptw.push_back(unit_root_neg((long long)t * j, Bp));
            Bp = S;
        }
        for (int pos = 0; pos < Nx; ++pos) {
            int rem = pos, m = 0, wgt = Nx;
            for (int q = P->prx.np - 1; q >= 0; --q) {     // digits from the last pass outwards
                const int rq = 1 << P->prx.lr[q];
                const int dgt = rem % rq;
                rem /= rq;
                wgt /= rq;
                m += dgt * wgt;
            }
            if (m == 0 || 2 * m == Nx) ikt[pos] = 0.0f;
            else {
                const int ms = (m <= Nx / 2) ? m : m - Nx;
                ikt[pos] = (float)(p->L / (2.0 * 3.14159265358979323846 * (double)ms * (double)Nx));
            }
        }
    }
    alloc((void**)&P->ikt, sizeof(float) * Nx);
    alloc((void**)&P->ptw, sizeof(float2) * ptw.size());
    P->ptw_len = (int)ptw.size();
    alloc((void**)&P->cg4, sizeof(float) * 4);
    float cg4h[4];
    for (int g = 0; g < 4; ++g) cg4h[g] = g < ng ? (float)p->feq.c[g] : 0.0f;
    alloc((void**)&P->os_lam_x, sizeof(float2) * OS_LAMW * (P->os_x ? Nv : 1));
    alloc((void**)&P->os_lam_v, sizeof(float2) * OS_LAMW * (P->os_v ? Nx + 16 : 1));   // rows of Nx + 16 entries
    alloc((void**)&P->taps_x, sizeof(float) * 32 * (P->os_x ? Nv : 1));
    alloc((void**)&P->taps_v, sizeof(float) * 32 * (P->os_v ? Nx + 16 : 1));
    alloc((void**)&P->xtwA, sizeof(float2) * xa.size());
    alloc((void**)&P->xtwB, sizeof(float2) * xb.size());
    alloc((void**)&P->xcs, sizeof(float2) * xc.size());
    alloc((void**)&P->rec_v, sizeof(float) * REC_WORDS * Nx);
    alloc((void**)&P->part, sizeof(double) * P->nby_max * Nx);
    alloc((void**)&P->partk, sizeof(double) * P->nby_max * Nx);
    alloc((void**)&P->diag, sizeof(double) * 8);
    alloc((void**)&P->rho, sizeof(double) * Nx);
    alloc((void**)&P->strip_flags, sizeof(int) * (Nx / 16 + 1));
    if (e == cudaSuccess) e = cudaMemsetAsync(P->strip_flags, 0, sizeof(int) * (Nx / 16 + 1), P->st);
    {
        int nsm = 0;
        int dev = 0;
        cudaGetDevice(&dev);
        cudaDeviceGetAttribute(&nsm, cudaDevAttrMultiProcessorCount, dev);
        if (nsm <= 0) nsm = 148;
        const size_t hb = sizeof(float) * (size_t)nsm * 4 * 2 * 40 * 16;
        alloc((void**)&P->ip_halo, hb);
        if (e == cudaSuccess) e = cudaMemsetAsync(P->ip_halo, 0, hb, P->st);
    }
    alloc((void**)&P->E_self, sizeof(float) * Nx);
    alloc((void**)&P->feq_tab, sizeof(float) * ((size_t)(ng ? ng : 1) * Nv + 512));   // + padding read (not used) by osv2_kernel
    if (e == cudaSuccess) e = cudaMemsetAsync(P->feq_tab, 0, sizeof(float) * ((size_t)(ng ? ng : 1) * Nv + 512), P->st);
    alloc((void**)&P->vmu_tab, sizeof(float) * (ng ? ng : 1) * Nv);
    if (e != cudaSuccess) { free_plan(P); cudaGetLastError(); return e == cudaErrorMemoryAllocation ? VOG_ENOMEM : VOG_ECUDA; }
    e = cudaMemcpyAsync(P->os_twv, otv.data(), sizeof(float2) * otv.size(), cudaMemcpyHostToDevice, P->st);
    if (e == cudaSuccess) e = cudaMemcpyAsync(P->cg4, cg4h, sizeof(cg4h), cudaMemcpyHostToDevice, P->st);
    if (e == cudaSuccess) e = cudaMemcpyAsync(P->ptw, ptw.data(), sizeof(float2) * ptw.size(), cudaMemcpyHostToDevice, P->st);
    if (e == cudaSuccess) e = cudaMemcpyAsync(P->ikt, ikt.data(), sizeof(float) * Nx, cudaMemcpyHostToDevice, P->st);
    if (e == cudaSuccess) e = cudaMemcpyAsync(P->os_cs64, ocs64.data(), sizeof(double2) * ocs64.size(), cudaMemcpyHostToDevice, P->st);
    if (e == cudaSuccess) e = cudaMemcpyAsync(P->xtwA, xa.data(), sizeof(float2) * xa.size(), cudaMemcpyHostToDevice, P->st);
    if (e == cudaSuccess) e = cudaMemcpyAsync(P->xtwB, xb.data(), sizeof(float2) * xb.size(), cudaMemcpyHostToDevice, P->st);
    if (e == cudaSuccess) e = cudaMemcpyAsync(P->xcs, xc.data(), sizeof(float2) * xc.size(), cudaMemcpyHostToDevice, P->st);
    if (e == cudaSuccess) e = cudaStreamSynchronize(P->st);
    std::vector<float2> h;
    fill_roots(h, Nx);
    if (e == cudaSuccess) e = cudaMemcpyAsync(P->tw_x, h.data(), sizeof(float2) * Nx, cudaMemcpyHostToDevice, P->st);
    if (e == cudaSuccess) e = cudaStreamSynchronize(P->st);
    fill_roots(h, Nv);
    if (e == cudaSuccess) e = cudaMemcpyAsync(P->tw_v, h.data(), sizeof(float2) * Nv, cudaMemcpyHostToDevice, P->st);
    if (e == cudaSuccess) e = cudaStreamSynchronize(P->st);
    if (ng > 0 && e == cudaSuccess) {
        std::vector<float> ft((size_t)ng * Nv), vt((size_t)ng * Nv);
        const double dv = (p->vmax - p->vmin) / (double)Nv;
        for (int g = 0; g < ng; ++g)
            for (int j = 0; j < Nv; ++j) {
                const double v = p->vmin + (double)j * dv;
                const double u = v - p->feq.mu[g];
                const double fe = p->feq.amp[g] * std::exp(-p->feq.c[g] * u * u);
                ft[(size_t)g * Nv + j] = (float)fe;
                vt[(size_t)g * Nv + j] = (float)u;
                P->feq_mass += dv * fe;
                P->feq_kin += 0.5 * p->L * dv * v * v * fe;
            }
        e = cudaMemcpyAsync(P->feq_tab, ft.data(), sizeof(float) * ft.size(), cudaMemcpyHostToDevice, P->st);
        if (e == cudaSuccess) e = cudaMemcpyAsync(P->vmu_tab, vt.data(), sizeof(float) * vt.size(), cudaMemcpyHostToDevice, P->st);
        if (e == cudaSuccess) e = cudaStreamSynchronize(P->st);
    }
    if (e == cudaSuccess && ((P->os_v && Nx / 16 <= P->n_sm) || Nx >= 4096)) {
        // steps solve the field in x space (field_then_v): inside the v kernel where it runs one piece per CTA, by
        // green_field_kernel on grids of 4096 columns or more
        e = cudaMalloc((void**)&P->green, sizeof(double) * Nx);
        // e_part: [Nx / 16] strip sums of E^2 | 1 word: ticket of the energy reduction | [Nx / 32] tickets of the density kernel
        if (e == cudaSuccess) e = cudaMalloc((void**)&P->e_part, sizeof(double) * (Nx / 16 + 1) + sizeof(unsigned) * (Nx / 32));
        if (e == cudaSuccess) e = cudaMemsetAsync(P->e_part, 0, sizeof(double) * (Nx / 16 + 1) + sizeof(unsigned) * (Nx / 32), P->st);
        std::vector<double> gh;
        green_host(Nx, p->L, gh);
        if (e == cudaSuccess) e = cudaMemcpyAsync(P->green, gh.data(), sizeof(double) * Nx, cudaMemcpyHostToDevice, P->st);
        if (e == cudaSuccess) e = cudaStreamSynchronize(P->st);
        if (e == cudaSuccess) P->fuse_field = 1;
        else { free_plan(P); cudaGetLastError(); return e == cudaErrorMemoryAllocation ? VOG_ENOMEM : VOG_ECUDA; }
    }
    if (e != cudaSuccess) { free_plan(P); cudaGetLastError(); return VOG_ECUDA; }
    *out = P;
    return VOG_OK;
}

extern "C" int vog_destroy(vog_plan_t P)
{
    if (!P) return VOG_EINVAL;
    cudaStreamSynchronize(P->st);
    free_plan(P);
    return VOG_OK;
}

// geometry of the overlap-save x launch for `lpi` lines per group (shared by vog_plan_tune and run_osx)
struct OsxShape { int np, thr, rounds; size_t smem6, smem7; };
static OsxShape osx_shape(const vog_plan_s* P, int lpi)
{
    OsxShape o;
    const int V = P->os_geom ? OS_VL : OS_V, tmax = 288;   // (launch bound of the x kernels)
    const int nb = (P->p.Nx + V - 1) / V;
    o.np = (nb + 1) / 2;
    const int pairs = o.np * lpi;
    o.rounds = 1;
    int per = pairs;
    while (16 * per > tmax) { ++o.rounds; per = (pairs + o.rounds - 1) / o.rounds; }
    o.thr = ((16 * per + 31) / 32) * 32;
    // bulk-landed kernel: lines (+ repeated head), two symbol rows per line, exchange scratch per resident pair
    o.smem6 = (size_t)lpi * (P->p.Nx + 480) * 4 + (size_t)2 * lpi * OS_LAMW * 8 + (size_t)(o.thr / 16) * (16 * 17 * 8) + 16;
    // warp-private windows (one round only): window slot, exchange scratch (overlapping by its unused last element) and
    // two shift words per pair, two symbol rows per line, one mbarrier per warp + 2
    o.smem7 = (size_t)(o.thr / 16) * (492 * 4 + (16 * 17 - 1) * 8 + 8) + 8 + (size_t)2 * lpi * OS_LAMW * 8 + (size_t)(o.thr / 32 + 2) * 8;
    return o;
}

// internal tuning hook (launch shapes only; results never change beyond rounding); codes in include/vog.h
extern "C" int vog_plan_tune(vog_plan_t P, int which, int value)
{
    if (!P) return VOG_EINVAL;
    const int Nx = P->p.Nx, Nv = P->p.Nv;
    switch (which) {
        case 2: if (value < 0 || (2 << value) > Nx || advect_smem_bytes(Nv, value) > 227 * 1024) return VOG_EINVAL; P->lognl_v = value; break;
        case 3: if (value < 32 || value > 512 || value % 32) return VOG_EINVAL; P->thr_v = value; break;
        case 5: if (value < 0 || (1 << value) > Nv || advect_x_smem_bytes(Nx, value, P->x_nbuf) > 227 * 1024) return VOG_EINVAL; P->x_lpi_log = value; P->x_occ = 0; break;
        case 6: if (value < 32 || value > 128 || value % 32) return VOG_EINVAL; P->x_thr = value; P->x_occ = 0; break;
        case 7: if (value < 0 || value > 32) return VOG_EINVAL; P->x_cps = value; break;
        case 8: if (value < 1 || value > 2 || advect_x_smem_bytes(Nx, P->x_lpi_log, value) > 227 * 1024) return VOG_EINVAL; P->x_nbuf = value; P->x_occ = 0; break;
        case 18: {
            if (value < 1 || value > Nv || !P->os_x) return VOG_EINVAL;
            const OsxShape o = osx_shape(P, value);
            if (((P->osx_variant == 0 && o.rounds == 1) ? o.smem7 : o.smem6) > 227 * 1024) return VOG_EINVAL;
            P->os2x_lpi = value; P->os3x_occ = 0; break;
        }
        case 20: if (value < 0) return VOG_EINVAL; P->os2v_gpc = value; break;
        case 21: {
            if (value < 0 || value > 1 || !P->os_x) return VOG_EINVAL;
            const OsxShape o = osx_shape(P, P->os2x_lpi);
            if (((value == 0 && o.rounds == 1) ? o.smem7 : o.smem6) > 227 * 1024) return VOG_EINVAL;
            P->osx_variant = value; P->os3x_occ = 0; break;
        }
        case 22: if (value < 0 || value > 2 || !P->os_v) return VOG_EINVAL; P->osv_variant = value; break;
        case 24: if (value < 1 || value > P->nby_max || (value & (value - 1)) || Nv / value < 32) return VOG_EINVAL; P->nby = value; break;
        case 25: if (value < 0 || value > 1 || (value == 1 && P->p.kind != VOG_LAGRANGE)) return VOG_EINVAL; P->os_geom = value; P->os3x_occ = 0; break;
        case 26: if (value < 0 || value > 1) return VOG_EINVAL; P->pdl = value; break;
        case 30: if (value < 0 || value > 1 || (value == 1 && !P->green)) return VOG_EINVAL; P->fuse_field = value; break;
        case 31: if (value < 0 || value > 1) return VOG_EINVAL; P->v_spec = value; break;
        case 33: if (value < 0 || value > 1) return VOG_EINVAL; P->density_pdl = value; break;
        case 34: if (value < 0 || value > 1) return VOG_EINVAL; P->v_inplace = value; break;
        case 29: if (value < 0 || value > 1 || P->p.Nx > 256 || P->p.Nv > 256) return VOG_EINVAL; P->small_run = value; break;
        case 28: if (value < 0 || value > 2) return VOG_EINVAL; P->solver = value; P->E_of = nullptr; P->E_valid = false; break;
        case 27: if (value < 0 || value > 1) return VOG_EINVAL; P->method = value; P->recx_valid = false; P->E_of = nullptr; break;
        default: return VOG_EINVAL;
    }
    return VOG_OK;
}

static int cuda_status(cudaError_t e)
{
    if (e == cudaSuccess) return VOG_OK;
    if (e == cudaErrorMemoryAllocation) { cudaGetLastError(); return VOG_ENOMEM; }
    return VOG_ECUDA;
}

static cudaError_t run_setup(vog_plan_s* P, bool vdir, int mode, double dt, const float* E, const float* Eext,
                             const double* beta)
{
    const int Nx = P->p.Nx, Nv = P->p.Nv;
    const double dv = (P->p.vmax - P->p.vmin) / (double)Nv;
    P->launches++;
    if (vdir ? P->os_v : P->os_x) {
        OsSetupArgs s;
        std::memset(&s, 0, sizeof(s));
        s.n_lines = vdir ? Nx : Nv;
        s.N = vdir ? Nv : Nx;
        s.mode = mode;
        s.spline = P->sym == SYM_SPLINE3;
        s.d = P->d;
        s.vdir = vdir ? 1 : 0;
        s.ks = Nx + 16;
        s.dt = dt; s.dv = dv;
        s.delta = vdir ? dv : P->p.L / (double)Nx;
        s.vmin = P->p.vmin;
        s.E = E; s.Eext = Eext; s.beta = beta;
        s.cs64 = P->os_cs64;
        s.lam = vdir ? P->os_lam_v : P->os_lam_x;
        if (P->method == 1) return st_setup_launch(s, vdir ? P->taps_v : P->taps_x, P->st);
        if (vdir && P->osv_variant == 0) {         // the default v kernel computes its strips' tables itself (S1 fused)
            P->vsetup = s;
            P->launches--;
            return cudaSuccess;
        }
        return os_setup_launch(s, P->st);
    }
    SetupArgs s;
    s.n_lines = vdir ? Nx : Nv;
    s.N = vdir ? Nv : Nx;
    s.mode = mode;
    s.spline = P->sym == SYM_SPLINE3;
    s.d = P->d;
    s.dt = dt;
    s.dv = dv;
    s.delta = vdir ? s.dv : P->p.L / (double)Nx;
    s.vmin = P->p.vmin;
    s.E = E; s.Eext = Eext; s.beta = beta;
    s.rec = vdir ? P->rec_v : P->xrec;
    if (vdir) return launch_pdl(shift_setup_kernel, dim3((s.n_lines + 127) / 128), dim3(128), 0, P->st, s);
    return launch_pdl(shift_setup_x_kernel, dim3((s.n_lines + 127) / 128), dim3(128), 0, P->st, s);
}

// ---- overlap-save launches (line length >= 1024; kernels in vog_os2.cuh)
static cudaError_t run_osx(vog_plan_s* P, const float* src, float* dst)
{
    OsArgs a;
    std::memset(&a, 0, sizeof(a));
    const int Nx = P->p.Nx, Nv = P->p.Nv;
    a.src = src; a.dst = dst; a.Nx = Nx; a.Nv = Nv; a.N = Nx;
    const int geom = P->os_geom;
    const OsxShape o = osx_shape(P, P->os2x_lpi);
    a.np = o.np;
    a.nb = 2 * o.np;
    a.inv_np = (65536u + (unsigned)a.np - 1u) / (unsigned)a.np;
    a.lam = P->os_lam_x; a.tw = P->os_twv;
    a.lpi = P->os2x_lpi;
    a.n_lines = Nv;
    a.n_groups = (Nv + a.lpi - 1) / a.lpi;
    // per-pair windows when the group fits one round of the CTA, whole lines otherwise (16384-cell lines) or on request
    const bool windows = P->osx_variant == 0 && o.rounds == 1;
    const size_t smem = windows ? o.smem7 : o.smem6;
    if (P->os3x_occ == 0) {
        P->os3x_occ = windows ? osx7_occupancy(geom, o.thr, smem) : osx6_occupancy(geom, o.thr, smem);
        if (P->os3x_occ <= 0) return cudaErrorInvalidConfiguration;
    }
    int grid = P->os3x_occ * P->n_sm;
    if (grid > a.n_groups) grid = a.n_groups;
    P->launches++;
    if (windows) return osx7_launch(a, geom, grid, o.thr, smem, P->st);
    return osx6_launch(a, geom, grid, o.thr, smem, P->st);
}

// ---- direct-stencil launches (line length >= 1024; kernels in vog_stencil.cu)
static cudaError_t run_stx(vog_plan_s* P, const float* src, float* dst)
{
    OsArgs a;
    std::memset(&a, 0, sizeof(a));
    const int Nx = P->p.Nx, Nv = P->p.Nv;
    a.src = src; a.dst = dst; a.Nx = Nx; a.Nv = Nv; a.N = Nx;
    a.np = Nx / 512;                               // segments per line
    int lpi = 256 / (16 * a.np);
    if (lpi < 1) lpi = 1;
    while (lpi > 1 && (Nv + lpi - 1) / lpi < P->n_sm * 3) --lpi;
    a.lpi = lpi;
    a.n_lines = Nv;
    a.n_groups = (Nv + lpi - 1) / lpi;
    const int thr = ((16 * a.np * lpi + 31) / 32) * 32;
    const int spline = P->sym == SYM_SPLINE3;
    const size_t smem = stx_smem_bytes(spline, P->d, thr);
    if (P->stx_occ == 0) {
        P->stx_occ = stx_occupancy(spline, P->d, thr, smem);
        if (P->stx_occ <= 0) return cudaErrorInvalidConfiguration;
    }
    int grid = P->stx_occ * P->n_sm;
    if (grid > a.n_groups) grid = a.n_groups;
    P->launches++;
    return stx_launch(a, spline, P->d, P->taps_x, grid, thr, smem, P->st);
}

static cudaError_t run_stv(vog_plan_s* P, const float* src, float* dst, bool source)
{
    OsArgs a;
    std::memset(&a, 0, sizeof(a));
    const int Nx = P->p.Nx, Nv = P->p.Nv;
    a.src = src; a.dst = dst; a.Nx = Nx; a.Nv = Nv; a.N = Nv;
    a.lam_ks = Nx + 16;
    a.ng = source ? P->p.feq.n : 0;
    a.feq_tab = P->feq_tab; a.vmu_tab = P->vmu_tab; a.cg4 = P->cg4;
    a.dvf = (float)((P->p.vmax - P->p.vmin) / (double)Nv);
    P->launches++;
    return stv_launch(a, P->sym == SYM_SPLINE3, P->d, P->taps_v, P->st);
}

static cudaError_t run_osv(vog_plan_s* P, const float* src, float* dst, bool source)
{
    OsArgs a;
    std::memset(&a, 0, sizeof(a));
    const int Nx = P->p.Nx, Nv = P->p.Nv;
    a.src = src; a.dst = dst; a.Nx = Nx; a.Nv = Nv; a.N = Nv;
    const int geom = P->os_geom;
    const int V = geom ? OS_VL : OS_V;
    a.nb = (Nv + V - 1) / V;
    a.np = (a.nb + 1) / 2;
    a.lam = P->os_lam_v; a.tw = P->os_twv; a.lam_ks = Nx + 16;
    a.ng = source ? P->p.feq.n : 0;
    a.feq_tab = P->feq_tab; a.vmu_tab = P->vmu_tab; a.cg4 = P->cg4;
    a.dvf = (float)((P->p.vmax - P->p.vmin) / (double)Nv);
    P->launches++;
    if (P->osv_variant == 0) {
        // three groups per CTA on one strip's symbol table; a work item is a segment of gpc consecutive pairs of a strip
        // (each group: every third pair of it, the next one's rows in flight while the current one is transformed)
        int gpc = P->os2v_gpc > 0 ? P->os2v_gpc : (a.np >= 18 ? 9 : (a.np >= 6 ? 3 : a.np));
        if (gpc > a.np) gpc = a.np;
        a.gpc = gpc;
        // (the first windows may be requested before the kernel's wait only when the kernel in front of it on the
        // stream is not the one that writes src: true behind a field solve, whose kernels only read the grid)
        P->vsetup.spec = P->v_spec && P->v_behind_field;
        a.inplace = P->v_inplace_now ? 1 : 0;
        a.dst2 = P->g_buf; a.strip_flags = P->strip_flags;
        a.halo = P->ip_halo;
        return osv7_launch(a, P->vsetup, geom, P->n_sm, P->st);
    }
    if (P->osv_variant == 2) {
        // 16-column strips, one group per CTA, symbol through L1
        int gpc = P->os2v_gpc > 0 ? P->os2v_gpc : (a.np >= 12 ? 3 : 1);
        if (gpc > a.np) gpc = a.np;
        a.gpc = gpc;
        return osv6_launch(a, geom, dim3(Nx / 16, (a.np + gpc - 1) / gpc), P->st);
    }
    const int strips = Nx / 32;
    int gpc = P->os2v_gpc > 0 ? P->os2v_gpc : 1;
    if (gpc > a.np) gpc = a.np;
    a.gpc = gpc;
    dim3 grid(strips, (a.np + gpc - 1) / gpc);
    return osv4_launch(a, geom, grid, 512, (size_t)256 * 32 * 8 + (size_t)OS_LAMW * 32 * 8 + 240 * 8 + 4 * 32 * 16, P->st);
}

static cudaError_t run_advect_x(vog_plan_s* P, float* f)
{
    AdvectXArgs a;
    const int Nx = P->p.Nx, Nv = P->p.Nv;
    a.f = f;
    a.lpi_log = P->x_lpi_log;
    a.nbuf = P->x_nbuf;
    a.n_groups = Nv >> a.lpi_log;
    a.twA = P->xtwA; a.twB = P->xtwB; a.cs = P->xcs; a.rec = P->xrec;
    for (int j = 0; j < 32; ++j) {
        const float2 w = unit_root_neg(j, 32);
        a.root32[j] = make_float2(w.x, -w.y);
    }
    const size_t smem = advect_x_smem_bytes(Nx, a.lpi_log, a.nbuf);
    if (P->x_occ == 0) {
        P->x_occ = advect_x_occupancy(Nx, P->sym, P->x_thr, smem);
        if (P->x_occ <= 0) return cudaErrorInvalidConfiguration;
    }
    const int cps = (P->x_cps > 0 && P->x_cps < P->x_occ) ? P->x_cps : P->x_occ;
    int grid = cps * P->n_sm;
    if (grid > a.n_groups) grid = a.n_groups;
    advect_x_launch_fn fn = advect_x_launcher(Nx);
    if (!fn) return cudaErrorInvalidValue;
    P->launches++;
    return fn(a, P->sym, grid, P->x_thr, smem, P->st);
}

static cudaError_t run_advect_line(vog_plan_s* P, float* f, bool vdir, bool source)
{
    if (!vdir) return run_advect_x(P, f);
    AdvectArgs a;
    std::memset(&a, 0, sizeof(a));
    const int Nx = P->p.Nx, Nv = P->p.Nv;
    const int N = vdir ? Nv : Nx, n_lines = vdir ? Nx : Nv;
    const int lognl = vdir ? P->lognl_v : P->lognl_x;
    a.f = f; a.Nx = Nx; a.Nv = Nv;
    a.tw = vdir ? P->tw_v : P->tw_x;
    a.rec = vdir ? P->rec_v : P->rec_x;
    a.lognl = lognl;
    a.ng = (vdir && source) ? P->p.feq.n : 0;
    a.feq_tab = P->feq_tab; a.vmu_tab = P->vmu_tab;
    for (int g = 0; g < 4; ++g) a.cg[g] = g < P->p.feq.n ? (float)P->p.feq.c[g] : 0.0f;
    const int n_tiles = n_lines / (2 << lognl);
    advect_launch_fn fn = advect_launcher(N);
    if (!fn) return cudaErrorInvalidValue;
    P->launches++;
    return fn(a, P->sym, vdir, n_tiles, vdir ? P->thr_v : P->thr_x, advect_smem_bytes(N, lognl), P->st);
}

static cudaError_t ensure_gbuf(vog_plan_s* P)
{
    if (P->g_buf) return cudaSuccess;
    return cudaMalloc((void**)&P->g_buf, sizeof(float) * (size_t)P->p.Nx * P->p.Nv);
}

static cudaError_t copy_grid(vog_plan_s* P, float* dst, const float* src)
{
    return cudaMemcpyAsync(dst, src, sizeof(float) * (size_t)P->p.Nx * P->p.Nv, cudaMemcpyDeviceToDevice, P->st);
}

// x-advection src -> dst (dst may equal src); the shift records/tables must be current
static cudaError_t advect_x(vog_plan_s* P, const float* src, float* dst)
{
    if (P->os_x) return P->method == 1 ? run_stx(P, src, dst) : run_osx(P, src, dst);
    cudaError_t e = cudaSuccess;
    if (src != dst) e = copy_grid(P, dst, src);
    if (e == cudaSuccess) e = run_advect_line(P, dst, false, false);
    return e;
}

// v-advection src -> dst; the overlap-save kernel needs dst != src, the whole-line kernel works in place
static cudaError_t advect_v(vog_plan_s* P, const float* src, float* dst, bool source)
{
    if (P->os_v) return src == dst ? cudaErrorInvalidValue : (P->method == 1 ? run_stv(P, src, dst, source) : run_osv(P, src, dst, source));
    cudaError_t e = cudaSuccess;
    if (src != dst) e = copy_grid(P, dst, src);
    if (e == cudaSuccess) e = run_advect_line(P, dst, true, source);
    return e;
}

// in-place v-advection through the plan's second grid buffer when the kernel is out of place
static cudaError_t advect_v_inplace(vog_plan_s* P, float* f, bool source)
{
    if (!P->os_v) return run_advect_line(P, f, true, source);
    cudaError_t e = ensure_gbuf(P);
    if (e == cudaSuccess && P->method == 0 && P->osv_variant == 0 && P->v_inplace) {
        // whole strips per CTA, stored in place where the integer shifts stay inside the kernel's saved halo (<= 24 rows);
        // the other strips go through the second grid and are copied back by a second, otherwise empty, launch
        P->v_inplace_now = true;
        e = run_osv(P, f, f, source);
        P->v_inplace_now = false;
        if (e == cudaSuccess) { e = strip_copy_launch(f, P->g_buf, P->strip_flags, P->p.Nx, P->p.Nv, P->st); P->launches++; }
        return e;
    }
    if (e == cudaSuccess) e = P->method == 1 ? run_stv(P, f, P->g_buf, source) : run_osv(P, f, P->g_buf, source);
    if (e == cudaSuccess) e = copy_grid(P, f, P->g_buf);
    return e;
}

static cudaError_t run_field(vog_plan_s* P, const float* f, float* E_out, double* energy_out = nullptr,
                             double* diag_out = nullptr)
{
    const int Nx = P->p.Nx, Nv = P->p.Nv;
    const double dv = (P->p.vmax - P->p.vmin) / (double)Nv, dx = P->p.L / (double)Nx;
    dim3 grid(Nx / 32, P->nby);
    cudaError_t e;
    const bool pdl_was = t_pdl;
    t_pdl = pdl_was && P->density_pdl;
    if (diag_out)
        e = launch_pdl(density_partial_kernel<true>, grid, dim3(256), 0, P->st, f, Nx, Nv, Nv / P->nby, P->part, P->partk,
                       P->p.vmin, dv, (unsigned*)nullptr, (double*)nullptr, 0.0);
    else
        e = launch_pdl(density_partial_kernel<false>, grid, dim3(256), 0, P->st, f, Nx, Nv, Nv / P->nby, P->part,
                       (double*)nullptr, 0.0, 0.0, (unsigned*)nullptr, (double*)nullptr, 0.0);
    t_pdl = pdl_was;
    if (e != cudaSuccess) return e;
    P->launches += 2;
    P->E_valid = true;
    P->E_of = f;
    int Ta = Nx < 1024 ? Nx : 1024;
    if (P->solver == 0) {
        int T = Nx / 4;                            // (radix-8 passes keep Nx / 8 threads busy, the loads and stores all)
        if (T > 1024) T = 1024;
        if (T < 32) T = 32;
        const int tw_in_smem = Nx <= 8192;
        const size_t psmem = sizeof(float2) * (Nx + Nx / 16) + sizeof(float) * Nx + (tw_in_smem ? sizeof(float2) * P->ptw_len : 0);
        e = set_max_smem((const void*)poisson_kernel, psmem);
        if (e != cudaSuccess) return e;
        e = launch_pdl(poisson_kernel, dim3(1), dim3(T), psmem, P->st, Nx, P->prx, P->ptw_len, tw_in_smem,
                       (const float2*)P->ptw, (const float*)P->ikt, (const double*)P->part, P->nby, dv, P->rho, P->E_self, E_out,
                       energy_out, 0.5 * dx);
        if (e != cudaSuccess || !diag_out) return e;
        P->launches++;
        return launch_pdl(field_aux_kernel, dim3(1), dim3(Ta), 0, P->st, Nx, 0, (const double*)P->part, (const double*)P->partk,
                          P->nby, dv, dx, 0.0, P->feq_mass, P->feq_kin, P->rho, P->E_self, (float*)nullptr, diag_out);
    }
    // trapezoid solve; the electric energy of vog_run goes through the plan's diagnostics scratch
    double* const dg = diag_out ? diag_out : (energy_out ? P->diag : nullptr);
    e = launch_pdl(field_aux_kernel, dim3(1), dim3(Ta), 0, P->st, Nx, P->solver, (const double*)P->part,
                   (const double*)(diag_out ? P->partk : nullptr), P->nby, dv, dx, 1.0 - P->feq_mass, P->feq_mass, P->feq_kin,
                   P->rho, P->E_self, E_out, dg);
    if (e == cudaSuccess && energy_out)
        e = cudaMemcpyAsync(energy_out, dg, sizeof(double), cudaMemcpyDeviceToDevice, P->st);
    return e;
}

// field solve from src, then the v-advection src -> dst over dts with E + E_ext (S8, S9, S1-S7).  On grids whose default
// v kernel runs one piece per CTA (Nx / 16 <= SMs) the Poisson launch is dropped: the density kernel's slab sums go
// straight to the v kernel, where every CTA computes E on its own 16 columns as the circular convolution of rho with the
// Green's function of the same Fourier solve (fp64) and the strip's first CTA publishes rho, E_self and the energy share.
static cudaError_t field_then_v(vog_plan_s* P, const float* src, float* dst, double dts, const float* Eext,
                                double* energy_out)
{
    const int Nx = P->p.Nx, Nv = P->p.Nv;
    const double dv = (P->p.vmax - P->p.vmin) / (double)Nv;
    const bool xspace = P->fuse_field && P->green && P->solver == 0;
    const bool fuse = xspace && Nx / 16 <= P->n_sm && P->os_v && P->method == 0 && P->osv_variant == 0 && src != dst;
    cudaError_t e;
    if (xspace && !fuse && Nx >= 4096) {
        // density (its last blocks write rho) -> green_field_kernel (E_self, energy) -> v-advection
        const bool pdl_was = t_pdl;
        t_pdl = pdl_was && P->density_pdl;
        e = launch_pdl(density_partial_kernel<false>, dim3(Nx / 32, P->nby), dim3(256), 0, P->st, src, Nx, Nv, Nv / P->nby,
                       P->part, (double*)nullptr, 0.0, 0.0, reinterpret_cast<unsigned*>(P->e_part + Nx / 16 + 1), P->rho, dv);
        t_pdl = pdl_was;
        if (e != cudaSuccess) return e;
        const size_t gsmem = sizeof(float) * ((size_t)Nx + Nx / 8 + Nx + 128) + sizeof(double) * 32 * 64;
        e = set_max_smem((const void*)green_field_kernel, gsmem);
        if (e != cudaSuccess) return e;
        e = launch_pdl(green_field_kernel, dim3(Nx / 64), dim3(1024), gsmem, P->st, Nx, (const double*)P->green,
                       (const double*)P->rho, P->E_self, energy_out, P->e_part,
                       reinterpret_cast<unsigned*>(P->e_part + Nx / 16), 0.5 * P->p.L / (double)Nx);
        if (e != cudaSuccess) return e;
        P->launches += 2;
        P->E_valid = true;
        P->E_of = src;
        e = run_setup(P, true, 1, dts, P->E_self, Eext, nullptr);
        P->v_behind_field = true;
        if (e == cudaSuccess) e = advect_v(P, src, dst, true);
        P->v_behind_field = false;
        return e;
    }
    if (!fuse) {
        e = run_field(P, src, nullptr, energy_out);
        if (e == cudaSuccess) e = run_setup(P, true, 1, dts, P->E_self, Eext, nullptr);
        P->v_behind_field = true;
        if (e == cudaSuccess) e = advect_v(P, src, dst, true);
        P->v_behind_field = false;
        return e;
    }
    const bool pdl_was = t_pdl;
    t_pdl = pdl_was && P->density_pdl;
    e = launch_pdl(density_partial_kernel<false>, dim3(Nx / 32, P->nby), dim3(256), 0, P->st, src, Nx, Nv, Nv / P->nby,
                   P->part, (double*)nullptr, 0.0, 0.0, reinterpret_cast<unsigned*>(P->e_part + Nx / 16 + 1), P->rho, dv);
    t_pdl = pdl_was;
    if (e != cudaSuccess) return e;
    P->launches++;
    P->E_valid = true;
    P->E_of = src;
    e = run_setup(P, true, 1, dts, P->E_self, Eext, nullptr);          // (records the shift source; no launch)
    if (e != cudaSuccess) return e;
    OsSetupArgs& su = P->vsetup;
    su.fpart = P->rho; su.green = P->green; su.nby = P->nby;
    su.E_out = P->E_self; su.rho_out = nullptr;
    su.energy_out = energy_out; su.e_part = P->e_part;
    su.ticket = reinterpret_cast<unsigned*>(P->e_part + Nx / 16);
    su.half_dx = 0.5 * P->p.L / (double)Nx;
    P->v_behind_field = true;
    e = run_osv(P, src, dst, true);
    P->v_behind_field = false;
    su.fpart = nullptr;
    return e;
}

static cudaError_t ensure_recx(vog_plan_s* P, double dt)
{
    if (P->recx_valid && P->recx_dt == dt) return cudaSuccess;
    cudaError_t e = run_setup(P, false, 0, dt, nullptr, nullptr, nullptr);
    P->recx_valid = (e == cudaSuccess);
    P->recx_dt = dt;
    return e;
}

extern "C" int vog_advect_x(vog_plan_t P, float* f_dev, double dt)
{
    if (!P || !f_dev || !std::isfinite(dt)) return VOG_EINVAL;
    t_pdl = P->pdl != 0;
    P->E_of = nullptr;                            // the state changes: the cached field no longer belongs to it
    cudaError_t e = ensure_recx(P, dt);
    if (e == cudaSuccess) e = advect_x(P, f_dev, f_dev);
    return cuda_status(e);
}

extern "C" int vog_advect_v(vog_plan_t P, float* f_dev, const float* E_dev, double dt)
{
    if (!P || !f_dev || !E_dev || !std::isfinite(dt)) return VOG_EINVAL;
    t_pdl = P->pdl != 0;
    P->E_of = nullptr;                            // the state changes: the cached field no longer belongs to it
    cudaError_t e = run_setup(P, true, 1, dt, E_dev, nullptr, nullptr);
    if (e == cudaSuccess) e = advect_v_inplace(P, f_dev, true);
    return cuda_status(e);
}

extern "C" int vog_shift_x(vog_plan_t P, float* f_dev, const double* beta)
{
    if (!P || !f_dev || !beta) return VOG_EINVAL;
    t_pdl = P->pdl != 0;
    P->E_of = nullptr;                            // the state changes: the cached field no longer belongs to it
    P->recx_valid = false;
    cudaError_t e = run_setup(P, false, 2, 0.0, nullptr, nullptr, beta);
    if (e == cudaSuccess) e = advect_x(P, f_dev, f_dev);
    return cuda_status(e);
}

extern "C" int vog_shift_v(vog_plan_t P, float* f_dev, const double* beta)
{
    if (!P || !f_dev || !beta) return VOG_EINVAL;
    t_pdl = P->pdl != 0;
    P->E_of = nullptr;                            // the state changes: the cached field no longer belongs to it
    cudaError_t e = run_setup(P, true, 2, 0.0, nullptr, nullptr, beta);
    if (e == cudaSuccess) e = advect_v_inplace(P, f_dev, false);
    return cuda_status(e);
}

extern "C" int vog_shift_v_to(vog_plan_t P, const float* src_dev, float* dst_dev, const double* beta)
{
    if (!P || !src_dev || !dst_dev || !beta || src_dev == dst_dev) return VOG_EINVAL;
    t_pdl = P->pdl != 0;
    P->E_of = nullptr;                            // the state changes: the cached field no longer belongs to it
    cudaError_t e = run_setup(P, true, 2, 0.0, nullptr, nullptr, beta);
    if (e == cudaSuccess) e = advect_v(P, src_dev, dst_dev, false);
    return cuda_status(e);
}

extern "C" int vog_field(vog_plan_t P, const float* f_dev, float* E_dev)
{
    if (!P || !f_dev || !E_dev) return VOG_EINVAL;
    t_pdl = P->pdl != 0;
    return cuda_status(run_field(P, f_dev, E_dev));
}

extern "C" int vog_diagnostics(vog_plan_t P, const float* f_dev, double* diag_dev)
{
    if (!P || !f_dev || !diag_dev) return VOG_EINVAL;
    t_pdl = P->pdl != 0;
    return cuda_status(run_field(P, f_dev, nullptr, nullptr, diag_dev));
}

extern "C" int vog_get_field(vog_plan_t P, float* E_dev)
{
    if (!P || !E_dev || !P->E_valid) return VOG_EINVAL;
    return cuda_status(cudaMemcpyAsync(E_dev, P->E_self, sizeof(float) * P->p.Nx, cudaMemcpyDeviceToDevice, P->st));
}

extern "C" int vog_step(vog_plan_t P, float* f_dev, double dt, const float* E_ext_dev)
{
    if (!P || !f_dev || !std::isfinite(dt)) return VOG_EINVAL;
    t_pdl = P->pdl != 0;
    cudaError_t e = cudaSuccess;
    // The overlap-save v kernel is out of place: it writes the plan's second grid g, and the x-advection
    // that follows reads g and writes f, so a step moves no extra bytes.
    float* g = f_dev;
    if (P->os_v) {
        e = ensure_gbuf(P);
        if (e != cudaSuccess) { cudaGetLastError(); return VOG_ENOMEM; }
        g = P->g_buf;
    }
    if (P->p.split == VOG_SPLIT_XVX) {
        e = ensure_recx(P, 0.5 * dt);
        if (e == cudaSuccess) e = advect_x(P, f_dev, f_dev);
        if (e == cudaSuccess) e = field_then_v(P, f_dev, g, dt, E_ext_dev, nullptr);
        if (e == cudaSuccess) e = advect_x(P, g, f_dev);
        P->E_of = nullptr;                        // E_self is the field at the half step, not of the final state
    } else {
        // E_prev: the field the previous VXV step on this array ended with; anything else is solved from f
        if (P->E_of != f_dev) e = run_field(P, f_dev, nullptr);
        if (e == cudaSuccess) e = run_setup(P, true, 1, 0.5 * dt, P->E_self, E_ext_dev, nullptr);
        if (e == cudaSuccess) e = advect_v(P, f_dev, g, true);
        if (e == cudaSuccess) e = ensure_recx(P, dt);
        if (e == cudaSuccess) e = advect_x(P, g, g);
        if (e == cudaSuccess) e = field_then_v(P, g, f_dev, 0.5 * dt, E_ext_dev, nullptr);
        P->E_of = e == cudaSuccess ? f_dev : nullptr;      // rho, hence E, is invariant under the v-advection
    }
    return cuda_status(e);
}

extern "C" int vog_run(vog_plan_t P, float* f_dev, double dt, int nsteps, const float* E_ext_seq_dev, int merge,
                       double* energy_dev)
{
    if (!P || !f_dev || nsteps < 0 || !std::isfinite(dt) || merge < 0 || merge > 1) return VOG_EINVAL;
    if (nsteps == 0) return VOG_OK;
    t_pdl = P->pdl != 0;
    const int Nx = P->p.Nx;
    cudaError_t e = cudaSuccess;
    if (P->small_run && P->solver == 0) {
        // the whole run as ONE persistent cluster kernel (vog_small.cu; vog_plan_tune(29, 1)): same sequences
        vog::SmallArgs a;
        const int Nv = P->p.Nv, C = vog::small_run_cluster(Nx, Nv);
        a.f = f_dev; a.E_out = P->E_self;
        a.E_init = (P->p.split == VOG_SPLIT_VXV && P->E_of == f_dev) ? P->E_self : nullptr;
        a.E_ext_seq = E_ext_seq_dev; a.energy = energy_dev;
        a.Nx = Nx; a.Nv = Nv; a.rpc = Nv / C;
        a.split = P->p.split; a.merge = merge; a.nsteps = nsteps;
        a.spline = P->p.kind == VOG_BSPLINE; a.d = a.spline ? 0 : (P->p.order - 1) / 2; a.ng = P->p.feq.n;
        a.dt = dt; a.L = P->p.L; a.vmin = P->p.vmin; a.dv = (P->p.vmax - P->p.vmin) / (double)Nv; a.dx = P->p.L / (double)Nx;
        for (int g = 0; g < 4; ++g) {
            a.amp[g] = P->p.feq.amp[g]; a.mu[g] = P->p.feq.mu[g]; a.c[g] = P->p.feq.c[g];
            a.cg[g] = g < a.ng ? (float)P->p.feq.c[g] : 0.0f;
        }
        e = vog::small_run_launch(a, P->st);
        P->launches++;
        P->E_valid = e == cudaSuccess;
        P->E_of = (e == cudaSuccess && P->p.split == VOG_SPLIT_VXV) ? f_dev : nullptr;
        return cuda_status(e);
    }
    float* g = f_dev;
    if (P->os_v) {
        e = ensure_gbuf(P);
        if (e != cudaSuccess) { cudaGetLastError(); return VOG_ENOMEM; }
        g = P->g_buf;
    }
    int iv = 0, ie = 0;                                    // v-advections and field solves so far
    auto ext = [&]() { return E_ext_seq_dev ? E_ext_seq_dev + (size_t)(iv++) * Nx : nullptr; };
    auto en = [&]() { return energy_dev ? energy_dev + (ie++) : nullptr; };
    auto ok = [&]() { return e == cudaSuccess; };
    if (P->p.split == VOG_SPLIT_XVX) {
        // x(dt/2) [field v(dt) x(dt)]^(n-1) field v(dt) x(dt/2); unmerged: the x(dt) is two x(dt/2)
        e = ensure_recx(P, 0.5 * dt);
        if (ok()) e = advect_x(P, f_dev, f_dev);
        for (int s = 0; s < nsteps && ok(); ++s) {
            e = field_then_v(P, f_dev, g, dt, ext(), en());
            const bool last = s == nsteps - 1;
            if (ok()) e = ensure_recx(P, (merge && !last) ? dt : 0.5 * dt);
            if (ok()) e = advect_x(P, g, f_dev);
            if (ok() && !merge && !last) e = advect_x(P, f_dev, f_dev);
        }
        P->E_of = nullptr;
    } else {
        // v(dt/2) [x(dt) field v(dt)]^(n-1) x(dt) field v(dt/2); the two v(dt/2) around a field solve see the same
        // E (rho is invariant under the v-advection), so merged they are one v(dt)
        float *cur = f_dev, *oth = g;                      // (oth == cur for the in-place whole-line kernels)
        auto vadv = [&](double dts) {
            e = run_setup(P, true, 1, dts, P->E_self, ext(), nullptr);
            if (ok()) e = advect_v(P, cur, oth, true);
            std::swap(cur, oth);
        };
        const int nvadv = merge ? nsteps + 1 : 2 * nsteps;
        bool flip_x = oth != cur && (nvadv & 1);           // odd number of buffer flips: one x-advection goes across
        if (P->E_of != f_dev) e = run_field(P, f_dev, nullptr, nullptr);
        if (ok()) vadv(0.5 * dt);
        if (ok()) e = ensure_recx(P, dt);
        for (int s = 0; s < nsteps && ok(); ++s) {
            if (flip_x) { e = advect_x(P, cur, oth); std::swap(cur, oth); flip_x = false; }
            else e = advect_x(P, cur, cur);
            const bool last = s == nsteps - 1;
            if (!ok()) break;
            // (field solve + the v-advection that follows it; unmerged, the second v(dt/2) reuses E_self)
            e = field_then_v(P, cur, oth, (merge && !last) ? dt : 0.5 * dt, ext(), en());
            std::swap(cur, oth);
            if (ok() && !(merge && !last) && !last) vadv(0.5 * dt);
        }
        P->E_of = ok() ? f_dev : nullptr;
    }
    return cuda_status(e);
}

static int run_host(vog_plan_t P, float* f_host, double dt, int nsteps, const float* E_ext_host, float* E_host, bool sync)
{
    if (!P || !f_host || nsteps < 0 || !std::isfinite(dt)) return VOG_EINVAL;
    const size_t nf = (size_t)P->p.Nx * P->p.Nv;
    cudaError_t e = cudaSuccess;
    if (!P->f_buf) {                                       // both buffers or neither
        float *fb = nullptr, *eb = nullptr;
        e = cudaMalloc((void**)&fb, sizeof(float) * nf);
        if (e == cudaSuccess) e = cudaMalloc((void**)&eb, sizeof(float) * P->p.Nx);
        if (e != cudaSuccess) { cudaFree(fb); cudaGetLastError(); return VOG_ENOMEM; }
        P->f_buf = fb; P->ext_buf = eb;
    }
    P->E_of = nullptr;                                    // new data in the staging buffer
    e = cudaMemcpyAsync(P->f_buf, f_host, sizeof(float) * nf, cudaMemcpyHostToDevice, P->st);
    if (e == cudaSuccess && E_ext_host)
        e = cudaMemcpyAsync(P->ext_buf, E_ext_host, sizeof(float) * P->p.Nx, cudaMemcpyHostToDevice, P->st);
    if (e != cudaSuccess) return VOG_ECUDA;
    for (int s = 0; s < nsteps; ++s) {
        int rc = vog_step(P, P->f_buf, dt, E_ext_host ? P->ext_buf : nullptr);
        if (rc != VOG_OK) return rc;
    }
    e = cudaMemcpyAsync(f_host, P->f_buf, sizeof(float) * nf, cudaMemcpyDeviceToHost, P->st);
    if (e == cudaSuccess && E_host && P->E_valid)
        e = cudaMemcpyAsync(E_host, P->E_self, sizeof(float) * P->p.Nx, cudaMemcpyDeviceToHost, P->st);
    if (e == cudaSuccess && sync) e = cudaStreamSynchronize(P->st);
    return cuda_status(e);
}

extern "C" int vog_run_host(vog_plan_t P, float* f_host, double dt, int nsteps, const float* E_ext_host, float* E_host)
{
    return run_host(P, f_host, dt, nsteps, E_ext_host, E_host, true);
}

extern "C" int vog_run_host_async(vog_plan_t P, float* f_host, double dt, int nsteps, const float* E_ext_host,
                                  float* E_host)
{
    return run_host(P, f_host, dt, nsteps, E_ext_host, E_host, false);
}

extern "C" int vog_reset(vog_plan_t P)
{
    if (!P) return VOG_EINVAL;
    P->E_valid = false;
    P->E_of = nullptr;
    P->recx_valid = false;
    return VOG_OK;
}

#ifdef VOG_STAMPS
extern "C" int vog_debug_stamps(long long* out32) { return (int)cudaMemcpyFromSymbol(out32, vog::vog_stamps, sizeof(long long) * 32); }
#endif

extern "C" long long vog_launch_count(vog_plan_t P) { return P ? P->launches + vog::f64_launches(P->f64) : -1; }

// ---- double-precision mode (NEXT-2; kernels and state in vog_f64.cu)
static int f64_state(vog_plan_s* P)
{
    if (P->f64) return VOG_OK;
    return vog::f64_create(&P->f64, &P->p, P->st, P->n_sm);
}
#define VOG_F64_ENTER(...) \
    if (!P || __VA_ARGS__) return VOG_EINVAL; \
    { const int rc = f64_state(P); if (rc != VOG_OK) return rc; }

extern "C" int vog_shift_x_f64(vog_plan_t P, double* f_dev, const double* beta)
{
    VOG_F64_ENTER(!f_dev || !beta)
    return cuda_status(vog::f64_shift(P->f64, f_dev, beta, false));
}
extern "C" int vog_shift_v_f64(vog_plan_t P, double* f_dev, const double* beta)
{
    VOG_F64_ENTER(!f_dev || !beta)
    return cuda_status(vog::f64_shift(P->f64, f_dev, beta, true));
}
extern "C" int vog_advect_x_f64(vog_plan_t P, double* f_dev, double dt)
{
    VOG_F64_ENTER(!f_dev || !std::isfinite(dt))
    return cuda_status(vog::f64_advect_x(P->f64, f_dev, dt));
}
extern "C" int vog_advect_v_f64(vog_plan_t P, double* f_dev, const double* E_dev, double dt)
{
    VOG_F64_ENTER(!f_dev || !E_dev || !std::isfinite(dt))
    return cuda_status(vog::f64_advect_v(P->f64, f_dev, E_dev, dt));
}
extern "C" int vog_field_f64(vog_plan_t P, const double* f_dev, double* E_dev)
{
    VOG_F64_ENTER(!f_dev || !E_dev)
    return cuda_status(vog::f64_field(P->f64, f_dev, E_dev));
}
extern "C" int vog_get_field_f64(vog_plan_t P, double* E_dev)
{
    if (!P || !E_dev || !vog::f64_has_field(P->f64)) return VOG_EINVAL;
    return cuda_status(vog::f64_get_field(P->f64, E_dev));
}
extern "C" int vog_step_f64(vog_plan_t P, double* f_dev, double dt, const double* E_ext_dev)
{
    VOG_F64_ENTER(!f_dev || !std::isfinite(dt))
    return cuda_status(vog::f64_step(P->f64, f_dev, dt, E_ext_dev));
}
