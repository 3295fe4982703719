// vog_small.cu -- the whole run of a SMALL grid (Nx, Nv <= 256) as ONE persistent kernel (SURVEY.md 8(f) NEXT-1:
// "persistent whole-step kernel").  Grids of 64^2 .. 256^2 are launch-bound: five launches per Strang
// step cost 24-35 us for a few microseconds of work.  Here the grid lives in the shared memory of a thread-block cluster
// (C = 1 .. 8 CTAs, Nv / C velocity rows each, two buffers) for all nsteps: x-advections are CTA-local, the density is
// reduced through distributed shared memory, every CTA solves its share of the Poisson problem, and the v-advection
// reads the rows it needs from its neighbours' shared memory.  Nothing goes to global memory between the first load and
// the last store except the optional energy history.
// Arithmetic: the circulant product of eq (4) in its direct form u'_i = sum_j a_j u_(i+b+j), taps in fp64 ->
// fp32 (the same matrix as the Fourier kernels up to rounding, like csrc/vog_stencil.cu; for 64..256-cell lines 18
// multiply-adds per cell cost no more than the transform); rho in fp64 in a fixed order; the Fourier solve of P:221 as
// two plain fp64 DFT sums split over the cluster; delta-f source with expm1f.  Sequences: exactly those of
// vog_run (both split orders, merge 0 / 1, E_ext per v-advection, energy per field solve).
// Selected per plan with vog_plan_tune(29, 1).  Product code; shares nothing with oracle/.
#include <cooperative_groups.h>
#include <cuda_runtime.h>

#include "vog_internal.h"

namespace cg = cooperative_groups;

namespace vog {

namespace sm {
constexpr int T = 512;                 // threads per CTA
constexpr int TW = 32;                 // floats per taps record (NT <= 29 taps; [30] source shift, [31] integer shift)
__host__ __device__ inline size_t smem_bytes(int Nx, int rpc)
{
    // doubles: part[Nx] rt[Nx] Ed[Nx] tw[2 Nx] Eh[Nx] red[T] wtab[32] | floats: bufA bufB tapsx[2][rpc][TW] tapsv[TW][Nx]
    // Ef[Nx] feqv[4][rpc] uu[4][rpc]
    return sizeof(double) * ((size_t)6 * Nx + T + 32) +
           sizeof(float) * ((size_t)2 * rpc * Nx + (size_t)2 * rpc * TW + (size_t)TW * Nx + Nx + 8 * (size_t)rpc);
}
}  // namespace sm

// four consecutive outputs from the register window r; M = misalignment of the first input (0..3)
template <int NT, int M>
__device__ __forceinline__ float4 small_dot4(const float* r, const float* w)
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

// taps of one line from its normalised displacement beta: integer shift b mod N, taps a_j, j = -JL .. NT-1-JL
// (Lagrange 2d+1: a_j = prod_{m != j} (b* - m) / (j - m) by prefix / suffix products and the constant
// 1 / prod (j - m) from wtab; cubic spline: a = m * g with g_n = wtab[n] = sqrt(3) (sqrt(3) - 2)^n).
template <int NT, int JL, class Put>
__device__ __forceinline__ int small_taps(const double beta, const int N, const int spline, const int d,
                                          const double* __restrict__ wtab, Put put)
{
    const double fl = floor(beta);
    const double t = beta - fl;
    int b;
    if (fabs(fl) < 9.0e18) {
        b = (int)(__double2ll_rn(fl) & (long long)(N - 1));
    } else {
        double bm = fmod(fl, (double)N);
        if (bm < 0.0) bm += (double)N;
        b = (int)bm;
        if (b >= N) b = 0;
    }
    if (!spline) {
        const int n = 2 * d + 2;
        double pre[18];
        double p = 1.0;
        for (int idx = 0; idx < n; ++idx) { pre[idx] = p; p *= t - (double)(idx - d); }
        for (int k = 0; k < NT; ++k)
            if (k < JL - d || k > JL + d + 1) put(k, 0.0);
        double sfx = 1.0;
        for (int idx = n - 1; idx >= 0; --idx) {
            put(idx - d + JL, pre[idx] * sfx * wtab[idx]);
            sfx *= t - (double)(idx - d);
        }
    } else {
        const double u = 1.0 - t;
        const double mq[4] = {u * u * u / 6.0, (4.0 - 6.0 * t * t + 3.0 * t * t * t) / 6.0,
                              (1.0 + 3.0 * t + 3.0 * t * t - 3.0 * t * t * t) / 6.0, t * t * t / 6.0};   // j = -1..2
        for (int k = 0; k < NT; ++k) {
            const int j = k - JL;
            double a = 0.0;
#pragma unroll
            for (int q = 0; q < 4; ++q) {
                const int nn = j - (q - 1);
                a += mq[q] * wtab[nn < 0 ? -nn : nn];
            }
            put(k, a);
        }
    }
    return b;
}

template <int NT, int JL>
__global__ void __launch_bounds__(sm::T, 1) small_run_kernel(const SmallArgs a)
{
    extern __shared__ __align__(16) unsigned char smem_raw[];
    cg::cluster_group cl = cg::this_cluster();
    const int rk = (int)cl.block_rank(), C = (int)cl.num_blocks();
    const int Nx = a.Nx, Nv = a.Nv, rpc = a.rpc, xmask = Nx - 1, vmask = Nv - 1;
    const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
    constexpr int T = sm::T, TW = sm::TW;
    // ---- shared memory (same offsets in every CTA of the cluster: remote addresses are formed from the local ones)
    double* const part = reinterpret_cast<double*>(smem_raw);     // [Nx] column sums of this CTA's rows
    double* const rt = part + Nx;                                  // [Nx] rho - mean
    double* const Ed = rt + Nx;                                    // [Nx] E (fp64), chunks written by their owners
    double2* const tw = reinterpret_cast<double2*>(Ed + Nx);       // [Nx] (cos, sin)(2 pi q / Nx)
    double2* const Eh = tw + Nx;                                   // [Nx / 2] E^_m, written by the modes' owners
    double* const red = reinterpret_cast<double*>(Eh + Nx / 2);    // [T]
    double* const wtab = red + T;                                  // [32]
    float* const bufA = reinterpret_cast<float*>(wtab + 32);       // [rpc][Nx]
    float* const bufB = bufA + (size_t)rpc * Nx;
    float* const tapsx = bufB + (size_t)rpc * Nx;                  // [2][rpc][TW]: dt/2, dt
    float* const tapsv = tapsx + 2 * rpc * TW;                     // [TW][Nx]
    float* const Ef = tapsv + TW * Nx;                             // [Nx] E rounded to fp32 (what vog_get_field returns)
    float* const feqv = Ef + Nx;                                   // [4][rpc] f_eq,g(v_j) of the local rows
    float* const uu = feqv + 4 * rpc;                              // [4][rpc] v_j - mu_g
    float* cur = bufA;
    float* oth = bufB;
    int lgx = 0, lgr = 0;
    while ((1 << lgx) < Nx) ++lgx;
    while ((1 << lgr) < rpc) ++lgr;

    auto csync = [&]() { cl.sync(); };             // (a cluster of one CTA: a block barrier)

    // ---- set-up: roots, constants of the taps, f_eq tables, x taps for dt/2 and dt, the CTA's rows of f
    for (int q = tid; q < Nx; q += T) {
        double sn, cs;
        sincospi(2.0 * (double)q / (double)Nx, &sn, &cs);
        tw[q] = make_double2(cs, sn);
    }
    if (tid < 32) {
        double w = 0.0;
        if (a.spline) {
            const double rt3 = 1.7320508075688772935;
            w = rt3 * pow(rt3 - 2.0, (double)tid);
        } else if (tid < 2 * a.d + 2) {
            const int j = tid - a.d;
            double den = 1.0;
            for (int m = -a.d; m <= a.d + 1; ++m)
                if (m != j) den *= (double)(j - m);
            w = 1.0 / den;
        }
        wtab[tid] = w;
    }
    for (int q = tid; q < 4 * rpc; q += T) {
        const int g = q / rpc, r = q - g * rpc;
        const double v = a.vmin + (double)(rk * rpc + r) * a.dv;
        double fe = 0.0, u = 0.0;
        if (g < a.ng) { u = v - a.mu[g]; fe = a.amp[g] * exp(-a.c[g] * u * u); }
        feqv[q] = (float)fe;
        uu[q] = (float)u;
    }
    __syncthreads();
    for (int q = tid; q < 2 * rpc; q += T) {
        const int w = q / rpc, r = q - w * rpc;
        const double dts = w == 0 ? 0.5 * a.dt : a.dt;
        const double beta = -(a.vmin + (double)(rk * rpc + r) * a.dv) * dts / a.dx;
        float* const rec = tapsx + (size_t)q * TW;
        const int b = small_taps<NT, JL>(beta, Nx, a.spline, a.d, wtab, [&](int k, double v) { rec[k] = (float)v; });
        rec[31] = __int_as_float(b);
    }
    {
        const float4* const src = reinterpret_cast<const float4*>(a.f + (size_t)rk * rpc * Nx);
        for (int q = tid; q < rpc * Nx / 4; q += T) reinterpret_cast<float4*>(cur)[q] = src[q];
    }
    csync();

    // ---- x-advection (rows are local): a warp takes (row, segment of 128 cells), a lane 4 consecutive cells from
    // 128-bit loads of the aligned window (misalignment M = (b - JL) mod 4, uniform over the row)
    auto X = [&](const int which) {
        constexpr int NCH = (NT + 9) / 4;
        const int segs = Nx > 128 ? Nx >> 7 : 1, cm = (Nx >> 2) - 1;
        for (int u = warp; u < rpc * segs; u += T / 32) {
            const int r = u / segs, sg = u - r * segs;
            const float* const rec = tapsx + (size_t)(which * rpc + r) * TW;
            const int bb = (__float_as_int(rec[31]) - JL) & xmask, M = bb & 3;
            const int c0 = 128 * sg + 4 * lane;
            if (c0 < Nx) {
                float w[NT];
#pragma unroll
                for (int k = 0; k < NT; ++k) w[k] = rec[k];
                const float4* const row4 = reinterpret_cast<const float4*>(cur + (size_t)r * Nx);
                const int ch0 = (c0 + bb - M) >> 2;
                float rg[4 * NCH];
#pragma unroll
                for (int n = 0; n < NCH; ++n) {
                    const float4 v = row4[(ch0 + n) & cm];
                    rg[4 * n] = v.x; rg[4 * n + 1] = v.y; rg[4 * n + 2] = v.z; rg[4 * n + 3] = v.w;
                }
                float4 o;
                switch (M) {
                    case 0: o = small_dot4<NT, 0>(rg, w); break;
                    case 1: o = small_dot4<NT, 1>(rg, w); break;
                    case 2: o = small_dot4<NT, 2>(rg, w); break;
                    default: o = small_dot4<NT, 3>(rg, w); break;
                }
                reinterpret_cast<float4*>(oth + (size_t)r * Nx)[c0 >> 2] = o;
            }
        }
        __syncthreads();
        float* const s = cur; cur = oth; oth = s;
    };

    // ---- field: rho (fp64, fixed order) -> zero mean -> E^_m = rho^_m / (i k_m), modes 0 and Nx/2 dropped -> E
    int ie = 0;
    auto F = [&](const bool with_energy) {
        {   // column sums of the local rows: T / Nx row lanes per column, folded in order
            const int parts = T >> lgx, i = tid & xmask, p = tid >> lgx;
            double s = 0.0;
            for (int r = p; r < rpc; r += parts) s += (double)cur[(size_t)r * Nx + i];
            red[tid] = s;
            __syncthreads();
            if (tid < Nx) {
                double t = 0.0;
                for (int q = 0; q < parts; ++q) t += red[q * Nx + tid];
                part[tid] = t;
            }
        }
        csync();
        double loc = 0.0;
        if (tid < Nx) {
            double t = 0.0;
            for (int q = 0; q < C; ++q) t += cl.map_shared_rank(part, q)[tid];      // ranks in order: deterministic
            loc = t * a.dv;
            rt[tid] = loc;
        }
#pragma unroll
        for (int o = 16; o > 0; o >>= 1) loc += __shfl_xor_sync(0xffffffffu, loc, o);
        __syncthreads();                           // (red is free again)
        if (lane == 0) red[warp] = loc;
        __syncthreads();
        double mean = 0.0;
        for (int w = 0; w < T / 32; ++w) mean += red[w];
        mean /= (double)Nx;
        if (tid < Nx) rt[tid] -= mean;
        __syncthreads();
        // forward sums: the modes 1 .. Nx/2 - 1 are dealt out over the cluster, one warp per mode
        const int nm = Nx / 2 - 1;
        for (int q = warp;; q += T / 32) {
            const int m = 1 + rk + C * q;
            if (m > nm) break;
            double sr = 0.0, si = 0.0;
            for (int i = lane; i < Nx; i += 32) {
                const double2 w = tw[(m * i) & xmask];
                const double r = rt[i];
                sr = fma(r, w.x, sr);
                si = fma(-r, w.y, si);
            }
#pragma unroll
            for (int o = 16; o > 0; o >>= 1) {
                sr += __shfl_xor_sync(0xffffffffu, sr, o);
                si += __shfl_xor_sync(0xffffffffu, si, o);
            }
            const double k = 2.0 * 3.14159265358979323846 * (double)m / a.L;
            if (lane < C) cl.map_shared_rank(Eh, lane)[m] = make_double2(si / k, -sr / k);   // (sr + i si) / (i k)
        }
        csync();
        // inverse sums: every CTA its chunk of cells, one warp per cell; E^_(Nx-m) = conj E^_m
        const int chunk = Nx / C;
        for (int q = warp; q < chunk; q += T / 32) {
            const int i = rk * chunk + q;
            double s = 0.0;
            for (int m = 1 + lane; m <= nm; m += 32) {
                const double2 w = tw[(m * i) & xmask];
                const double2 e = Eh[m];
                s += e.x * w.x - e.y * w.y;
            }
#pragma unroll
            for (int o = 16; o > 0; o >>= 1) s += __shfl_xor_sync(0xffffffffu, s, o);
            if (lane < C) cl.map_shared_rank(Ed, lane)[i] = 2.0 * s / (double)Nx;
        }
        csync();
        double e2 = 0.0;
        if (tid < Nx) {
            const float e = (float)Ed[tid];
            Ef[tid] = e;
            e2 = (double)e * (double)e;
        }
        if (with_energy && a.energy) {             // electric energy (1/2) dx sum E_i^2, fixed order
#pragma unroll
            for (int o = 16; o > 0; o >>= 1) e2 += __shfl_xor_sync(0xffffffffu, e2, o);
            if (lane == 0) red[warp] = e2;
            __syncthreads();
            if (rk == 0 && tid == 0) {
                double s = 0.0;
                for (int w = 0; w < T / 32; ++w) s += red[w];
                a.energy[ie] = 0.5 * a.dx * s;
            }
            ++ie;
        }
        __syncthreads();
    };

    // ---- v-advection over dts with the field E + E_ext (columns span the cluster): taps per column, then a thread
    // takes one column and 8 consecutive local rows from a sliding register window; the rows it reads may live in any
    // CTA of the cluster (distributed shared memory).  delta-f source with s = E dts.
    int iv = 0;
    auto V = [&](const double dts) {
        const float* const ext = a.E_ext_seq ? a.E_ext_seq + (size_t)iv * Nx : nullptr;
        ++iv;
        if (tid < Nx) {
            double e = (double)Ef[tid];
            if (ext) e += (double)ext[tid];
            const double beta = -e * dts / a.dv;
            const int b = small_taps<NT, JL>(beta, Nv, a.spline, a.d, wtab,
                                             [&](int k, double v) { tapsv[k * Nx + tid] = (float)v; });
            tapsv[30 * Nx + tid] = (float)(dts * e);
            tapsv[31 * Nx + tid] = __int_as_float(b);
        }
        __syncthreads();
        const int units = (rpc >> 3) << lgx;       // (column, group of 8 rows)
        for (int u = tid; u < units; u += T) {
            const int i = u & xmask, r0 = (u >> lgx) << 3;
            float w[NT];
#pragma unroll
            for (int k = 0; k < NT; ++k) w[k] = tapsv[k * Nx + i];
            const int j0 = rk * rpc + r0 + __float_as_int(tapsv[31 * Nx + i]) - JL;
            float acc[8];
#pragma unroll
            for (int r = 0; r < 8; ++r) acc[r] = 0.0f;
#pragma unroll
            for (int n = 0; n < NT + 7; ++n) {
                const int row = (j0 + n) & vmask;
                const float v = cl.map_shared_rank(cur, row >> lgr)[(size_t)(row & (rpc - 1)) * Nx + i];
#pragma unroll
                for (int r = 0; r < 8; ++r)
                    if (n - r >= 0 && n - r < NT) acc[r] = fmaf(w[n - r], v, acc[r]);
            }
            if (a.ng > 0) {
                const float s = tapsv[30 * Nx + i];
#pragma unroll
                for (int r = 0; r < 8; ++r) {
                    float q = 0.0f;
                    for (int g = 0; g < a.ng; ++g) {
                        const float ug = uu[g * rpc + r0 + r];
                        q = fmaf(feqv[g * rpc + r0 + r], expm1f(a.cg[g] * s * (2.0f * ug - s)), q);
                    }
                    acc[r] += q;
                }
            }
#pragma unroll
            for (int r = 0; r < 8; ++r) oth[(size_t)(r0 + r) * Nx + i] = acc[r];
        }
        csync();                                   // everybody has read its source rows and written its own
        float* const s = cur; cur = oth; oth = s;
    };

    // ---- the sequences of vog_run
    const int n = a.nsteps;
    if (a.split == VOG_SPLIT_XVX) {
        // x(dt/2) [field v(dt) x(dt)]^(n-1) field v(dt) x(dt/2); unmerged: the x(dt) is two x(dt/2)
        X(0);
        for (int s = 0; s < n; ++s) {
            F(true);
            V(a.dt);
            const bool last = s == n - 1;
            X((a.merge && !last) ? 1 : 0);
            if (!a.merge && !last) X(0);
        }
    } else {
        // v(dt/2) [x(dt) field v(dt)]^(n-1) x(dt) field v(dt/2)
        if (a.E_init) {
            if (tid < Nx) Ef[tid] = a.E_init[tid];
            __syncthreads();
        } else {
            F(false);
        }
        V(0.5 * a.dt);
        for (int s = 0; s < n; ++s) {
            X(1);
            F(true);
            const bool last = s == n - 1;
            if (a.merge && !last) V(a.dt);
            else {
                V(0.5 * a.dt);
                if (!last) V(0.5 * a.dt);
            }
        }
    }
    // ---- results
    {
        float4* const dst = reinterpret_cast<float4*>(a.f + (size_t)rk * rpc * Nx);
        for (int q = tid; q < rpc * Nx / 4; q += T) dst[q] = reinterpret_cast<const float4*>(cur)[q];
    }
    if (rk == 0 && a.E_out)
        for (int q = tid; q < Nx; q += T) a.E_out[q] = Ef[q];
    csync();                                       // no CTA leaves while its shared memory may still be read
}

// host: cluster size and launch
int small_run_cluster(int Nx, int Nv)
{
    int C = (Nx * Nv) / 8192;
    if (C < 1) C = 1;
    if (C > 8) C = 8;
    return C;
}

template <int NT, int JL>
static cudaError_t small_launch_t(const SmallArgs& a, int C, cudaStream_t st)
{
    const size_t smem = sm::smem_bytes(a.Nx, a.rpc);
    cudaError_t e = set_max_smem((const void*)small_run_kernel<NT, JL>, smem);
    if (e != cudaSuccess) return e;
    cudaLaunchConfig_t cfg = {};
    cfg.gridDim = dim3(C);
    cfg.blockDim = dim3(sm::T);
    cfg.dynamicSmemBytes = smem;
    cfg.stream = st;
    cudaLaunchAttribute at[1];
    at[0].id = cudaLaunchAttributeClusterDimension;
    at[0].val.clusterDim.x = C;
    at[0].val.clusterDim.y = 1;
    at[0].val.clusterDim.z = 1;
    cfg.attrs = at;
    cfg.numAttrs = 1;
    return cudaLaunchKernelEx(&cfg, small_run_kernel<NT, JL>, a);
}

cudaError_t small_run_launch(const SmallArgs& a, cudaStream_t st)
{
    const int C = a.Nv / a.rpc;
    if (a.spline) return small_launch_t<29, 14>(a, C, st);
    if (a.d <= 1) return small_launch_t<4, 1>(a, C, st);
    if (a.d <= 4) return small_launch_t<10, 4>(a, C, st);
    return small_launch_t<18, 8>(a, C, st);
}

}  // namespace vog
