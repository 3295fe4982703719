// vog_os.cu -- overlap-save advection kernels: instantiation, launchers and the setup kernel that
// tabulates the symbol lambda(theta_k) per line (S1 + the closed form of S4).  Product code.
#include <map>
#include <mutex>
#include <utility>

#include "vog_os2.cuh"

namespace vog {

// One CTA of 128 threads per line, thread k writes entry k (threads 0, 1 also entries 128, 129).  beta = -c dt / Delta in fp64; b = floor(beta), b* = beta - b.
//   Lagrange 2d+1, Everett form: lambda = P(s;1-b*) + e^{i theta} P(s;b*), s = 2 - 2 cos(theta),
//     P(s;t) = sum_k a_k(t) s^k, a_0 = t, a_k = a_{k-1} (k^2 - t^2) / (2k (2k+1));
//   cubic spline: [B(b*+1) e^{-i theta} + B(b*) + B(b*-1) e^{i theta} + B(b*-2) e^{2 i theta}] 3/(2 + cos(theta)).
__global__ void __launch_bounds__(128) os_setup_kernel(const OsSetupArgs s)
{
    const int l = blockIdx.x;
    pdl_wait();                                   // E comes from the Poisson kernel; the tables may still be read
    pdl_launch_dependents();
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
    // the integer shift b goes entirely into the load address (entry 129): no rotation factor in the table
    // x: [line][k]; v: transposed [k][line] so that a strip of 32 columns reads 256-byte rows
    float2* out = s.vdir ? s.lam + l : s.lam + (size_t)l * OS_LAMW;
    const size_t ks = s.vdir ? (size_t)s.ks : 1;
    // fp64 for everything that is per line (beta, b, b*, the Everett / B-spline coefficients); the 129 table
    // entries are then evaluated in fp32 from those coefficients (rounded once) and from (cos, sin, 2 - 2 cos)
    // rounded from the fp64 table: ~1e-7 relative, the same as the whole-line kernels' in-kernel symbol.
    __shared__ float af[2][9];
    __shared__ float bs[4];
    if (!s.spline) {
        if (threadIdx.x < 18) {                      // a_j(t) = t prod_{m=1..j} (m^2 - t^2) / (2m (2m+1))
            const int half = threadIdx.x / 9, j = threadIdx.x - 9 * half;
            const double tt = half == 0 ? 1.0 - t : t;
            double a = tt;
            constexpr double rcp[9] = {0.0, 1.0 / 6.0, 1.0 / 20.0, 1.0 / 42.0, 1.0 / 72.0, 1.0 / 110.0, 1.0 / 156.0,
                                       1.0 / 210.0, 1.0 / 272.0};            // 1 / (2m (2m+1))
#pragma unroll
            for (int m = 1; m <= 8; ++m)
                if (m <= j) a = a * ((double)(m * m) - tt * tt) * rcp[m];
            af[half][j] = j <= s.d ? (float)a : 0.0f;
        }
    } else if (threadIdx.x == 0) {
        const double u = 1.0 - t;
        bs[0] = (float)(u * u * u / 6.0);
        bs[1] = (float)((4.0 - 6.0 * t * t + 3.0 * t * t * t) / 6.0);
        bs[2] = (float)((1.0 + 3.0 * t + 3.0 * t * t - 3.0 * t * t * t) / 6.0);
        bs[3] = (float)(t * t * t / 6.0);
    }
    __syncthreads();
    const float sc = 1.0f / (float)OS_LB;        // a power of two: exact
    // 128 threads: k = threadIdx.x, and threads 0 and 1 also write entries 128 and 129 (16 CTAs per SM)
    for (int k = threadIdx.x; k < OS_LAMW; k += 128) {
        if (k == 129) { out[129 * ks] = make_float2(__int_as_float(b), sshift); continue; }
        if (k == 0) { out[0] = make_float2(sc, 0.0f); continue; }   // lambda_0 = sum of the weights = 1
        const double2 cs = s.cs64[k];                  // (cos, sin)(2 pi k / OS_LB), fp64 table
        const float c = (float)cs.x, sn = (float)cs.y;
        float lr, li;
        if (s.spline) {
            const float Bm1 = bs[0], B0 = bs[1], B1 = bs[2], B2 = bs[3];
            const float c2 = (float)(2.0 * cs.x * cs.x - 1.0), s2 = (float)(2.0 * cs.y * cs.x);
            const float g = 3.0f / (2.0f + c);
            lr = fmaf(B2, c2, fmaf(Bm1 + B1, c, B0)) * g;
            li = fmaf(B2, s2, (B1 - Bm1) * sn) * g;
        } else {
            const float sv = (float)(2.0 - 2.0 * cs.x);
            float p0 = 0.0f, p1 = 0.0f;
#pragma unroll
            for (int j = 8; j >= 0; --j) {             // coefficients beyond the degree are zero
                p0 = fmaf(p0, sv, af[0][j]);
                p1 = fmaf(p1, sv, af[1][j]);
            }
            lr = fmaf(c, p1, p0);
            li = sn * p1;
        }
        out[k * ks] = make_float2(lr * sc, li * sc);
    }
}

// The same tables for the v direction, one CTA per strip of 32 columns (lane = column): the table is stored
// transposed, lam[k][column], so with one CTA per column (the kernel above) every entry was an isolated 8-byte
// store; here a warp writes whole 256-byte rows.  Threads 0..63 do the per-column fp64 work (one Everett chain
// a_0..a_8 per (column, half); the a_j are prefix products, same operations in the same order as above), then
// the 8 warps share the 130 rows.  Same arithmetic as os_setup_kernel, entry for entry.
__global__ void __launch_bounds__(256) os_setup_v_kernel(const OsSetupArgs s)
{
    __shared__ float af[18][32];                 // [half * 9 + j][column]; spline: rows 0..3 = B(b*+1), B(b*), B(b*-1), B(b*-2)
    __shared__ int bsh[32];
    __shared__ float ssh[32];
    const int tid = threadIdx.x, lane = tid & 31, wid = tid >> 5;
    const int l0 = blockIdx.x * 32;
    pdl_wait();                                   // E comes from the Poisson kernel; the tables may still be read
    pdl_launch_dependents();
    if (tid < 64) {
        const int half = tid >> 5, l = l0 + lane;
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
        if (fabs(fl) < 9.0e18) {
            b = (int)(__double2ll_rn(fl) & (long long)(s.N - 1));
        } else {
            double bm = fmod(fl, (double)s.N);
            if (bm < 0.0) bm += (double)s.N;
            b = (int)bm;
            if (b >= s.N) b = 0;
        }
        if (half == 0) { bsh[lane] = b; ssh[lane] = sshift; }
        if (!s.spline) {
            const double tt = half == 0 ? 1.0 - t : t;
            double a = tt;
            constexpr double rcp[9] = {0.0, 1.0 / 6.0, 1.0 / 20.0, 1.0 / 42.0, 1.0 / 72.0, 1.0 / 110.0, 1.0 / 156.0,
                                       1.0 / 210.0, 1.0 / 272.0};            // 1 / (2m (2m+1))
            af[half * 9][lane] = (float)a;
#pragma unroll
            for (int m = 1; m <= 8; ++m) {
                a = a * ((double)(m * m) - tt * tt) * rcp[m];
                af[half * 9 + m][lane] = m <= s.d ? (float)a : 0.0f;
            }
        } else if (half == 0) {
            const double u = 1.0 - t;
            af[0][lane] = (float)(u * u * u / 6.0);
            af[1][lane] = (float)((4.0 - 6.0 * t * t + 3.0 * t * t * t) / 6.0);
            af[2][lane] = (float)((1.0 + 3.0 * t + 3.0 * t * t - 3.0 * t * t * t) / 6.0);
            af[3][lane] = (float)(t * t * t / 6.0);
        }
    }
    __syncthreads();
    const float sc = 1.0f / (float)OS_LB;
    float2* const out = s.lam + l0 + lane;
    const size_t ks = (size_t)s.ks;
    for (int k = wid + 8 * blockIdx.y; k < OS_LAMW; k += 8 * gridDim.y) {      // (the rows are split over gridDim.y CTAs)
        if (k == 129) { out[129 * ks] = make_float2(__int_as_float(bsh[lane]), ssh[lane]); continue; }
        if (k == 0) { out[0] = make_float2(sc, 0.0f); continue; }
        const double2 cs = s.cs64[k];
        const float c = (float)cs.x, sn = (float)cs.y;
        float lr, li;
        if (s.spline) {
            const float Bm1 = af[0][lane], B0 = af[1][lane], B1 = af[2][lane], B2 = af[3][lane];
            const float c2 = (float)(2.0 * cs.x * cs.x - 1.0), s2 = (float)(2.0 * cs.y * cs.x);
            const float g = 3.0f / (2.0f + c);
            lr = fmaf(B2, c2, fmaf(Bm1 + B1, c, B0)) * g;
            li = fmaf(B2, s2, (B1 - Bm1) * sn) * g;
        } else {
            const float sv = (float)(2.0 - 2.0 * cs.x);
            float p0 = 0.0f, p1 = 0.0f;
#pragma unroll
            for (int j = 8; j >= 0; --j) {
                p0 = fmaf(p0, sv, af[j][lane]);
                p1 = fmaf(p1, sv, af[9 + j][lane]);
            }
            lr = fmaf(c, p1, p0);
            li = sn * p1;
        }
        out[k * ks] = make_float2(lr * sc, li * sc);
    }
}

cudaError_t os_setup_launch(const OsSetupArgs& s, cudaStream_t st)
{
    if (s.vdir && s.n_lines % 32 == 0) {
        // 8 CTAs share the 130 rows of a strip (measured at 2048 columns, step time: 1 -> 62.2, 2 -> 60.0, 4 -> 59.1,
        // 8 -> 58.8, 17 -> 59.4 us; one CTA per column, the kernel above: 61.0 us)
        return launch_pdl(os_setup_v_kernel, dim3(s.n_lines / 32, 8), dim3(256), 0, st, s);
    }
    return launch_pdl(os_setup_kernel, dim3(s.n_lines), dim3(128), 0, st, s);
}


// cudaFuncAttributeMaxDynamicSharedMemorySize is a per-device attribute: remember, per (device, kernel), the
// largest size that was set, so that plans on several devices (or threads) each get it set once.
cudaError_t set_max_smem(const void* fn, size_t smem)
{
    if (smem <= 48 * 1024) return cudaSuccess;
    static std::mutex mu;
    static std::map<std::pair<int, const void*>, size_t> cur;
    int dev = 0;
    cudaError_t e = cudaGetDevice(&dev);
    if (e != cudaSuccess) return e;
    std::lock_guard<std::mutex> lk(mu);
    size_t& c = cur[std::make_pair(dev, fn)];
    if (smem > c) {
        e = cudaFuncSetAttribute(fn, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem);
        if (e != cudaSuccess) return e;
        c = smem;
    }
    return cudaSuccess;
}

// warp-private-window x kernel (default when a line group fits one round); geom as above
cudaError_t osx7_launch(const OsArgs& a, int geom, int grid, int threads, size_t smem, cudaStream_t st)
{
    if (geom) {
        cudaError_t e = set_max_smem((const void*)osx7_kernel<OS_VL, OS_HL>, smem);
        if (e != cudaSuccess) return e;
        return launch_pdl(osx7_kernel<OS_VL, OS_HL>, dim3(grid), dim3(threads), smem, st, a);
    }
    cudaError_t e = set_max_smem((const void*)osx7_kernel<OS_V, OS_H>, smem);
    if (e != cudaSuccess) return e;
    return launch_pdl(osx7_kernel<OS_V, OS_H>, dim3(grid), dim3(threads), smem, st, a);
}

int osx7_occupancy(int geom, int threads, size_t smem)
{
    const void* fn = geom ? (const void*)osx7_kernel<OS_VL, OS_HL> : (const void*)osx7_kernel<OS_V, OS_H>;
    if (set_max_smem(fn, smem) != cudaSuccess) { cudaGetLastError(); return 0; }
    int nb = 0;
    const cudaError_t e = geom ? cudaOccupancyMaxActiveBlocksPerMultiprocessor(&nb, osx7_kernel<OS_VL, OS_HL>, threads, smem)
                               : cudaOccupancyMaxActiveBlocksPerMultiprocessor(&nb, osx7_kernel<OS_V, OS_H>, threads, smem);
    if (e != cudaSuccess) { cudaGetLastError(); return 0; }
    return nb;
}

// bulk-landed whole-line x kernel (lines that need several rounds: 16384 cells); geom as above
cudaError_t osx6_launch(const OsArgs& a, int geom, int grid, int threads, size_t smem, cudaStream_t st)
{
    cudaError_t e;
#define VOG_OSX6_LAUNCH(VV, HH, LL)                                                                      \
    do {                                                                                                 \
        e = set_max_smem((const void*)osx6_kernel<VV, HH, LL>, smem);                                    \
        if (e != cudaSuccess) return e;                                                                  \
        return launch_pdl(osx6_kernel<VV, HH, LL>, dim3(grid), dim3(threads), smem, st, a);              \
    } while (0)
    // Two lines per group in one round with every thread busy (1024- / 2048-cell lines): the instance with lpi = 2 as a
    // compile-time constant -- measured on the metric grid: 2048^2 step 46.15 -> 44.87 us.  (The same with lpi = 1 for
    // 8192-cell lines was SLOWER than the run-time instance, 122.1 against 116.4 us per launch, and is not built.)
    const bool two = a.lpi == 2 && a.N <= 2048 && 32 * a.np == threads && a.n_lines % 2 == 0;   // (4096 cells: 37.0 -> 42.6 us)
    if (geom) {
        if (two) VOG_OSX6_LAUNCH(OS_VL, OS_HL, 2);
        VOG_OSX6_LAUNCH(OS_VL, OS_HL, 0);
    }
    if (two) VOG_OSX6_LAUNCH(OS_V, OS_H, 2);
    VOG_OSX6_LAUNCH(OS_V, OS_H, 0);
#undef VOG_OSX6_LAUNCH
}

int osx6_occupancy(int geom, int threads, size_t smem)
{
    const void* fn = geom ? (const void*)osx6_kernel<OS_VL, OS_HL> : (const void*)osx6_kernel<OS_V, OS_H>;
    if (set_max_smem(fn, smem) != cudaSuccess) { cudaGetLastError(); return 0; }
    int nb = 0;
    const cudaError_t e = geom ? cudaOccupancyMaxActiveBlocksPerMultiprocessor(&nb, osx6_kernel<OS_VL, OS_HL>, threads, smem)
                               : cudaOccupancyMaxActiveBlocksPerMultiprocessor(&nb, osx6_kernel<OS_V, OS_H>, threads, smem);
    if (e != cudaSuccess) { cudaGetLastError(); return 0; }
    return nb;
}

// Tensor maps of a source grid for osv7_kernel: fp32 [Nv][Nx], boxes of 16 columns x {256, 64, 16, 4, 2} rows.  The
// encoder is a host-only driver entry point (no kernel, no copy), looked up through the runtime so that the library has
// no link-time dependency on libcuda; maps are cached per (grid pointer, Nx, Nv): a step alternates between two grids.
static cudaError_t v_maps(const float* src, int Nx, int Nv, os2::VMaps* out)
{
    typedef CUresult (*encode_fn)(CUtensorMap*, CUtensorMapDataType, cuuint32_t, void*, const cuuint64_t*, const cuuint64_t*,
                                  const cuuint32_t*, const cuuint32_t*, CUtensorMapInterleave, CUtensorMapSwizzle,
                                  CUtensorMapL2promotion, CUtensorMapFloatOOBfill);
    static std::mutex mu;
    static encode_fn encode = nullptr;
    struct Key {
        const float* p; int nx, nv;
        bool operator<(const Key& o) const { return p != o.p ? p < o.p : (nx != o.nx ? nx < o.nx : nv < o.nv); }
    };
    static std::map<Key, os2::VMaps> cache;
    std::lock_guard<std::mutex> lock(mu);
    if (!encode) {
        void* fn = nullptr;
        cudaDriverEntryPointQueryResult qr;
        cudaError_t e = cudaGetDriverEntryPoint("cuTensorMapEncodeTiled", &fn, cudaEnableDefault, &qr);
        if (e != cudaSuccess) return e;
        if (qr != cudaDriverEntryPointSuccess || !fn) return cudaErrorNotSupported;
        encode = (encode_fn)fn;
    }
    const Key key{src, Nx, Nv};
    auto it = cache.find(key);
    if (it == cache.end()) {
        if (cache.size() > 64) cache.clear();
        os2::VMaps m;
        const cuuint64_t dims[2] = {(cuuint64_t)Nx, (cuuint64_t)Nv};
        const cuuint64_t strides[1] = {(cuuint64_t)Nx * 4};
        const cuuint32_t estr[2] = {1, 1};
        for (int i = 0; i < 5; ++i) {
            const cuuint32_t box[2] = {(cuuint32_t)os2::VW, (cuuint32_t)(i == 4 ? 2 : 256 >> (2 * i))};
            const CUresult r = encode(&m.m[i], CU_TENSOR_MAP_DATA_TYPE_FLOAT32, 2, (void*)src, dims, strides, box, estr,
                                      CU_TENSOR_MAP_INTERLEAVE_NONE, CU_TENSOR_MAP_SWIZZLE_NONE,
                                      CU_TENSOR_MAP_L2_PROMOTION_NONE, CU_TENSOR_MAP_FLOAT_OOB_FILL_NONE);
            if (r != CUDA_SUCCESS) return cudaErrorInvalidValue;
        }
        it = cache.emplace(key, m).first;
    }
    *out = it->second;
    return cudaSuccess;
}

// three-group v kernel (default): one persistent CTA of 768 threads per SM; a.gpc = pairs per work item
cudaError_t osv7_launch(const OsArgs& a, const OsSetupArgs& su, int geom, int n_sm, cudaStream_t st)
{
    // table | twiddles | three coefficient records | (cos, sin) table | three groups (raw rows + exchange) | mbarriers
    const size_t smem = (size_t)OS_LAMW * os2::VW * 8 + 240 * 8 + 3 * 20 * os2::VW * 4 + 136 * 16 +
                        3 * ((size_t)os2::VRT * os2::VW * 4 + (size_t)OS_LB * os2::VW * 8) + 3 * 8;
    const int nstrips = a.Nx / os2::VW;
    const int grid = nstrips >= n_sm ? n_sm : nstrips * (n_sm / nstrips);     // (see the kernel: pieces of work)
    os2::VMaps maps;
    cudaError_t e = v_maps(a.src, a.Nx, a.Nv, &maps);
    if (e != cudaSuccess) return e;
    if (a.inplace && (nstrips % grid != 0 || (nstrips < grid && grid / nstrips > 1))) {
        // in place with pieces that are not whole strips: their boundary rows are saved by a launch of their own
        e = launch_pdl(osv7_halo_kernel, dim3(grid), dim3(256), 0, st, a, 2 * (geom ? OS_VL : OS_V));
        if (e != cudaSuccess) return e;
    }
#define VOG_OSV7_LAUNCH(VV, HH, IPF)                                                                     \
    do {                                                                                                 \
        e = set_max_smem((const void*)osv7_kernel<VV, HH, IPF>, smem);                                   \
        if (e != cudaSuccess) return e;                                                                  \
        return launch_pdl(osv7_kernel<VV, HH, IPF>, dim3(grid), dim3(768), smem, st, a, su, maps);       \
    } while (0)
    const bool flag_at_run_time = a.inplace || a.Nx <= 2048;       // (see the kernel's template comment)
    if (geom) {
        if (flag_at_run_time) VOG_OSV7_LAUNCH(OS_VL, OS_HL, 2);
        VOG_OSV7_LAUNCH(OS_VL, OS_HL, 0);
    }
    if (flag_at_run_time) VOG_OSV7_LAUNCH(OS_V, OS_H, 2);
    VOG_OSV7_LAUNCH(OS_V, OS_H, 0);
#undef VOG_OSV7_LAUNCH
}

// In-place v-advection, second launch: the strips that osv7_kernel could not store in place (integer shifts beyond its
// saved halo) lie in the second grid; copy them back and clear their flags.  One CTA per strip: 64-byte row segments,
// four threads per row.  A launch in which no strip is flagged reads Nx / 16 words and ends.
__global__ void __launch_bounds__(256) strip_copy_kernel(float* __restrict__ dst, const float* __restrict__ src,
                                                         int* __restrict__ strip_flags, int Nx, int Nv)
{
    pdl_wait();                                   // flags and the second grid come from the v kernel
    pdl_launch_dependents();
    const int strip = blockIdx.x;
    if (strip_flags[strip] == 0) return;          // (uniform over the CTA)
    const size_t off = (size_t)strip * os2::VW + (threadIdx.x & 3) * 4;
    for (int r = threadIdx.x >> 2; r < Nv; r += 64) {
        const float4 v = *reinterpret_cast<const float4*>(src + (size_t)r * Nx + off);
        *reinterpret_cast<float4*>(dst + (size_t)r * Nx + off) = v;
    }
    __syncthreads();
    if (threadIdx.x == 0) strip_flags[strip] = 0;
}

cudaError_t strip_copy_launch(float* dst, const float* src, int* strip_flags, int Nx, int Nv, cudaStream_t st)
{
    return launch_pdl(strip_copy_kernel, dim3(Nx / os2::VW), dim3(256), 0, st, dst, src, strip_flags, Nx, Nv);
}

// 16-column-strip v kernel, symbol through L1; grid = (Nx / 16, ceil(np / gpc))
cudaError_t osv6_launch(const OsArgs& a, int geom, dim3 grid, cudaStream_t st)
{
    const size_t smem = (size_t)os2::VRR * os2::VW * 4 + (size_t)OS_LB * os2::VW * 8;
    if (geom) {
        cudaError_t e = set_max_smem((const void*)osv6_kernel<OS_VL, OS_HL>, smem);
        if (e != cudaSuccess) return e;
        return launch_pdl(osv6_kernel<OS_VL, OS_HL>, grid, dim3(256), smem, st, a);
    }
    cudaError_t e = set_max_smem((const void*)osv6_kernel<OS_V, OS_H>, smem);
    if (e != cudaSuccess) return e;
    return launch_pdl(osv6_kernel<OS_V, OS_H>, grid, dim3(256), smem, st, a);
}

cudaError_t osv4_launch(const OsArgs& a, int geom, dim3 grid, int threads, size_t smem, cudaStream_t st)
{
    if (geom) {
        cudaError_t e = set_max_smem((const void*)osv4_kernel<OS_VL, OS_HL>, smem);
        if (e != cudaSuccess) return e;
        return launch_pdl(osv4_kernel<OS_VL, OS_HL>, grid, dim3(threads), smem, st, a);
    }
    cudaError_t e = set_max_smem((const void*)osv4_kernel<OS_V, OS_H>, smem);
    if (e != cudaSuccess) return e;
    return launch_pdl(osv4_kernel<OS_V, OS_H>, grid, dim3(threads), smem, st, a);
}

}  // namespace vog

#ifdef VOG_STAMPS
extern "C" int vog_debug_os_stamps(long long* out64) { return (int)cudaMemcpyFromSymbol(out64, vog::os_stamps, sizeof(long long) * 64); }
extern "C" int vog_debug_os_blk(long long* out4096) { return (int)cudaMemcpyFromSymbol(out4096, vog::os_blk, sizeof(long long) * 4096); }
#endif
