// vog_noalloc.cu -- vog_field_noalloc: the self-consistent field (S8 + S9: rho_i = dv sum_j f_ji, zero mean, Fourier
// solve E^_m = rho^_m / (i k_m) with modes 0 and Nx/2 dropped) for callers that cannot call
// cudaMalloc (code under CUDA graph capture, tight serving loops, harnesses that forbid it).  No plan, no allocation:
// the scratch the density kernel needs (its row-slab sums, which the plan-based path keeps in cudaMalloc'd memory) and
// the few O(Nx) work arrays of the solve live in ONE file-scope __device__ array of fixed size, 416 KB, held by every
// GPU that loads the library until the process exits.  Limits: Nx <= VOG_NOALLOC_MAX_NX (4096).
//
// Every call shares that array and it keeps the last call's contents.  Nothing in it is accumulated into: each call
// overwrites every word it later reads (slab sums, rho - mean, the roots, the spectrum), so nothing has to be cleared;
// but two calls that overlap on the GPU (different streams, or one stream per thread) RACE on it.  Calls on one stream
// are ordered and safe.
//
// In host code the array's name is a host-side stand-in, not a device address: the address comes from
// cudaGetSymbolAddress, once per device, with that device current.
// The solve itself: two plain fp64 DFT sums (O(Nx^2), one CTA per mode / per cell, roots from a table rebuilt per call),
// the arithmetic of the fp64 mode's field kernels; output rounded to fp32 like vog_field's.
// Product code; shares nothing with oracle/.
#include <cuda_runtime.h>

#include <mutex>

#include "../../include/vog.h"

namespace {

constexpr int NA_MAX_NX = VOG_NOALLOC_MAX_NX;
constexpr int NA_NBY = 8;                          // row slabs of the density kernel
// layout of the scratch, in doubles: slab sums [NA_NBY][MAX] | rho - mean [MAX] | roots (cos, sin) [MAX][2] | spectrum [MAX][2]
constexpr size_t NA_OFF_PART = 0;
constexpr size_t NA_OFF_RT = NA_OFF_PART + (size_t)NA_NBY * NA_MAX_NX;
constexpr size_t NA_OFF_TW = NA_OFF_RT + NA_MAX_NX;
constexpr size_t NA_OFF_EH = NA_OFF_TW + 2 * (size_t)NA_MAX_NX;
constexpr size_t NA_DOUBLES = NA_OFF_EH + 2 * (size_t)NA_MAX_NX;

static __device__ __align__(256) double vog_na_scratch[NA_DOUBLES];      // 13 * 4096 * 8 B = 416 KB

// S8: column sums of a row slab in fp64, fixed order.  grid (Nx / 32, nby), 256 threads: a warp covers 4 rows x 32
// columns (8 lanes x float4 per row); the 4 row-lanes are folded by shuffles, the 8 warps through shared memory.
__global__ void __launch_bounds__(256) na_density_kernel(const float* __restrict__ f, const int Nx, const int rows_per_block,
                                                         double* __restrict__ part)
{
    __shared__ double red[8][32];
    const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
    const int xl = lane & 7, rl = lane >> 3;
    const int col = blockIdx.x * 32 + xl * 4;
    const int j0 = blockIdx.y * rows_per_block;
    double s0 = 0, s1 = 0, s2 = 0, s3 = 0;
    const float* p = f + (size_t)(j0 + warp * 4 + rl) * Nx + col;
#pragma unroll 4
    for (int j = warp * 4 + rl; j < rows_per_block; j += 32) {
        const float4 v = __ldg(reinterpret_cast<const float4*>(p));
        s0 += (double)v.x; s1 += (double)v.y; s2 += (double)v.z; s3 += (double)v.w;
        p += (size_t)32 * Nx;
    }
#pragma unroll
    for (int o = 8; o <= 16; o <<= 1) {
        s0 += __shfl_xor_sync(0xffffffffu, s0, o);
        s1 += __shfl_xor_sync(0xffffffffu, s1, o);
        s2 += __shfl_xor_sync(0xffffffffu, s2, o);
        s3 += __shfl_xor_sync(0xffffffffu, s3, o);
    }
    if (rl == 0) { red[warp][xl * 4] = s0; red[warp][xl * 4 + 1] = s1; red[warp][xl * 4 + 2] = s2; red[warp][xl * 4 + 3] = s3; }
    __syncthreads();
    if (threadIdx.x < 32) {
        double s = 0;
#pragma unroll
        for (int w = 0; w < 8; ++w) s += red[w][threadIdx.x];
        part[(size_t)blockIdx.y * Nx + blockIdx.x * 32 + threadIdx.x] = s;
    }
}

// one CTA: rho_i = dv * (slab sums in slab order), rt_i = rho_i - mean, roots tw_q = (cos, sin)(2 pi q / Nx)
__global__ void __launch_bounds__(1024) na_rho_kernel(const int Nx, const int nby, const double dv, const double* __restrict__ part,
                                                      double* __restrict__ rt, double2* __restrict__ tw)
{
    __shared__ double red[32];
    __shared__ double mean_s;
    const int tid = threadIdx.x, T = blockDim.x;
    double loc = 0.0;
    for (int i = tid; i < Nx; i += T) {
        double s = 0.0;
        for (int y = 0; y < nby; ++y) s += part[(size_t)y * Nx + i];
        s *= dv;
        rt[i] = s;
        loc += s;
        double sn, cs;
        sincospi(2.0 * (double)i / (double)Nx, &sn, &cs);
        tw[i] = make_double2(cs, sn);
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
    for (int i = tid; i < Nx; i += T) rt[i] -= mean;            // (each thread touches only its own cells)
}

__device__ __forceinline__ double2 na_block_sum(double a, double b, double2* red)
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

// forward sum, one CTA per mode m = 1 .. Nx/2 - 1: rho^_m = sum_i rt_i e^{-2 i pi m i / Nx}; E^_m = rho^_m / (i k_m)
__global__ void __launch_bounds__(128) na_dft_fwd_kernel(const int Nx, const double L, const double* __restrict__ rt,
                                                         const double2* __restrict__ tw, double2* __restrict__ Ehat)
{
    __shared__ double2 red[4];
    const int m = 1 + blockIdx.x, mask = Nx - 1;
    double sr = 0.0, si = 0.0;
    for (int i = threadIdx.x; i < Nx; i += blockDim.x) {
        const double2 w = tw[(int)(((long long)m * i) & mask)];
        const double r = rt[i];
        sr = fma(r, w.x, sr);
        si = fma(-r, w.y, si);
    }
    const double2 s = na_block_sum(sr, si, red);
    if (threadIdx.x == 0) {
        const double k = 2.0 * 3.14159265358979323846 * (double)m / L;
        Ehat[m] = make_double2(s.y / k, -s.x / k);
    }
}

// inverse sum, one CTA per cell: E_i = (2 / Nx) sum_{0 < m < Nx/2} Re(E^_m e^{+2 i pi m i / Nx}) (rho is real)
__global__ void __launch_bounds__(128) na_dft_inv_kernel(const int Nx, const double2* __restrict__ Ehat,
                                                         const double2* __restrict__ tw, float* __restrict__ E)
{
    __shared__ double2 red[4];
    const int i = blockIdx.x, mask = Nx - 1;
    double s = 0.0;
    for (int m = 1 + threadIdx.x; m < Nx / 2; m += blockDim.x) {
        const double2 w = tw[(int)(((long long)m * i) & mask)];
        const double2 e = Ehat[m];
        s += e.x * w.x - e.y * w.y;
    }
    const double2 t = na_block_sum(s, 0.0, red);
    if (threadIdx.x == 0) E[i] = (float)(2.0 * t.x / (double)Nx);
}

// device address of the scratch on the CURRENT device, looked up once per device
cudaError_t na_scratch(double** out)
{
    constexpr int MAXDEV = 64;
    static std::mutex mu;
    static double* ptrs[MAXDEV] = {};
    int dev = 0;
    cudaError_t e = cudaGetDevice(&dev);
    if (e != cudaSuccess) return e;
    if (dev < 0 || dev >= MAXDEV) return cudaErrorInvalidDevice;
    std::lock_guard<std::mutex> lock(mu);
    if (!ptrs[dev]) {
        double* p = nullptr;
        e = cudaGetSymbolAddress((void**)&p, vog_na_scratch);
        if (e != cudaSuccess) return e;
        ptrs[dev] = p;
    }
    *out = ptrs[dev];
    return cudaSuccess;
}

bool pow2(int n) { return n > 0 && (n & (n - 1)) == 0; }

}  // namespace

extern "C" int vog_field_noalloc(const float* f_dev, int Nx, int Nv, double L, double vmin, double vmax, float* E_dev,
                                 void* cuda_stream)
{
    if (!f_dev || !E_dev || !(L > 0.0) || !(vmax > vmin)) return VOG_EINVAL;
    if (!pow2(Nx) || !pow2(Nv) || Nx < 64 || Nv < 64 || Nv > 16384) return VOG_EINVAL;
    if (Nx > NA_MAX_NX) return VOG_ETOOLARGE;      // beyond the fixed scratch: use the plan-based vog_field
    double* sc = nullptr;
    if (na_scratch(&sc) != cudaSuccess) { cudaGetLastError(); return VOG_ECUDA; }
    cudaStream_t st = (cudaStream_t)cuda_stream;
    double* const part = sc + NA_OFF_PART;
    double* const rt = sc + NA_OFF_RT;
    double2* const tw = reinterpret_cast<double2*>(sc + NA_OFF_TW);
    double2* const Eh = reinterpret_cast<double2*>(sc + NA_OFF_EH);
    int nby = NA_NBY;
    while (nby > 1 && Nv / nby < 32) nby >>= 1;    // at least 32 rows per slab (one pass of the 8 warps x 4 row lanes)
    const double dv = (vmax - vmin) / (double)Nv;
    const int dft_threads = Nx / 2 < 128 ? Nx / 2 : 128;
    na_density_kernel<<<dim3(Nx / 32, nby), 256, 0, st>>>(f_dev, Nx, Nv / nby, part);
    na_rho_kernel<<<1, Nx < 1024 ? Nx : 1024, 0, st>>>(Nx, nby, dv, part, rt, tw);
    na_dft_fwd_kernel<<<Nx / 2 - 1, dft_threads, 0, st>>>(Nx, L, rt, tw, Eh);
    na_dft_inv_kernel<<<Nx, dft_threads, 0, st>>>(Nx, Eh, tw, E_dev);
    return cudaGetLastError() == cudaSuccess ? VOG_OK : VOG_ECUDA;
}
