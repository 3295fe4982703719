// vog_advect_inst.cu -- instantiates the fused advection kernel for ONE line length
// (compile with -DVOG_N=<64..16384>; the build compiles this file once per length).
#include "vog_advect.cuh"
#include "vog_advect_x.cuh"

#ifndef VOG_N
#error "compile with -DVOG_N=<line length>"
#endif
#define VOG_CAT2(a, b) a##b
#define VOG_CAT(a, b) VOG_CAT2(a, b)

namespace vog {

template <int N, int SYM, bool VDIR>
static cudaError_t launch_one(const AdvectArgs& a, int n_tiles, int threads, size_t smem, cudaStream_t st)
{
    auto kern = advect_kernel<N, SYM, VDIR>;
    const cudaError_t e = set_max_smem((const void*)kern, smem);
    if (e != cudaSuccess) return e;
    return launch_pdl(kern, dim3(n_tiles), dim3(threads), smem, st, a);
}

template <int N, bool VDIR>
static cudaError_t launch_sym(const AdvectArgs& a, int sym, int n_tiles, int threads, size_t smem, cudaStream_t st)
{
    switch (sym) {
        case SYM_LAG_D1:  return launch_one<N, SYM_LAG_D1, VDIR>(a, n_tiles, threads, smem, st);
        case SYM_LAG_D4:  return launch_one<N, SYM_LAG_D4, VDIR>(a, n_tiles, threads, smem, st);
        case SYM_LAG_D8:  return launch_one<N, SYM_LAG_D8, VDIR>(a, n_tiles, threads, smem, st);
        case SYM_SPLINE3: return launch_one<N, SYM_SPLINE3, VDIR>(a, n_tiles, threads, smem, st);
    }
    return cudaErrorInvalidValue;
}

cudaError_t VOG_CAT(advect_launch_, VOG_N)(const AdvectArgs& a, int sym, bool vdir, int n_tiles, int threads,
                                           size_t smem, cudaStream_t st)
{
    // the contiguous direction is served by advect_x_kernel (vog_advect_x.cuh); only the column-tile
    // instantiation of this kernel is built
    return vdir ? launch_sym<VOG_N, true>(a, sym, n_tiles, threads, smem, st) : cudaErrorInvalidValue;
}

// ---- contiguous-line (x) kernel
template <int N, int SYM>
static cudaError_t launch_x_one(const AdvectXArgs& a, int grid, int threads, size_t smem, cudaStream_t st)
{
    auto kern = advect_x_kernel<N, SYM>;
    const cudaError_t e = set_max_smem((const void*)kern, smem);
    if (e != cudaSuccess) return e;
    return launch_pdl(kern, dim3(grid), dim3(threads), smem, st, a);
}

template <int N, int SYM>
static int occ_x_one(int threads, size_t smem)
{
    auto kern = advect_x_kernel<N, SYM>;
    if (set_max_smem((const void*)kern, smem) != cudaSuccess) {
        cudaGetLastError();
        return 0;
    }
    int nb = 0;
    if (cudaOccupancyMaxActiveBlocksPerMultiprocessor(&nb, kern, threads, smem) != cudaSuccess) {
        cudaGetLastError();
        return 0;
    }
    return nb;
}

cudaError_t VOG_CAT(advect_x_launch_, VOG_N)(const AdvectXArgs& a, int sym, int grid, int threads, size_t smem,
                                             cudaStream_t st)
{
    switch (sym) {
        case SYM_LAG_D1:  return launch_x_one<VOG_N, SYM_LAG_D1>(a, grid, threads, smem, st);
        case SYM_LAG_D4:  return launch_x_one<VOG_N, SYM_LAG_D4>(a, grid, threads, smem, st);
        case SYM_LAG_D8:  return launch_x_one<VOG_N, SYM_LAG_D8>(a, grid, threads, smem, st);
        case SYM_SPLINE3: return launch_x_one<VOG_N, SYM_SPLINE3>(a, grid, threads, smem, st);
    }
    return cudaErrorInvalidValue;
}

int VOG_CAT(advect_x_occ_, VOG_N)(int sym, int threads, size_t smem)
{
    switch (sym) {
        case SYM_LAG_D1:  return occ_x_one<VOG_N, SYM_LAG_D1>(threads, smem);
        case SYM_LAG_D4:  return occ_x_one<VOG_N, SYM_LAG_D4>(threads, smem);
        case SYM_LAG_D8:  return occ_x_one<VOG_N, SYM_LAG_D8>(threads, smem);
        case SYM_SPLINE3: return occ_x_one<VOG_N, SYM_SPLINE3>(threads, smem);
    }
    return 0;
}

}  // namespace vog
