// vog_internal.h -- structures shared by the translation units of libvog (product code only).
#pragma once
#include <cuda_runtime.h>

#include <utility>

#include "../../include/vog.h"

namespace vog {

// ---- Programmatic dependent launch.  The kernels of a Strang step (S1-S9) run back to back on one stream and at
// 2048^2 each lasts 7-23 us, so the drain / launch / ramp-up between two of them is a visible share of the step.
// A kernel launched with launch_pdl() may become resident while its predecessor in the stream is still running;
// it MUST call pdl_wait() before its first access to anything the predecessor reads or writes (the wait returns
// when the predecessor grid has completed and its memory is visible), and calls pdl_launch_dependents() so
// that its own successor may be staged early.  Work placed before pdl_wait() may only touch memory that is constant
// for the life of the plan (twiddle tables).
#ifdef __CUDACC__
__device__ __forceinline__ void pdl_wait() { asm volatile("griddepcontrol.wait;" ::: "memory"); }
__device__ __forceinline__ void pdl_launch_dependents() { asm volatile("griddepcontrol.launch_dependents;" ::: "memory"); }

bool pdl_enabled();   // vog_lib.cu: false when the environment holds VOG_NO_PDL=1 (A/B measurements)

template <typename... KArgs, typename... Args>
static inline cudaError_t launch_pdl(void (*kern)(KArgs...), dim3 grid, dim3 block, size_t smem, cudaStream_t st,
                                     Args&&... args)
{
    cudaLaunchConfig_t cfg = {};
    cfg.gridDim = grid;
    cfg.blockDim = block;
    cfg.dynamicSmemBytes = smem;
    cfg.stream = st;
    cudaLaunchAttribute at[1];
    at[0].id = cudaLaunchAttributeProgrammaticStreamSerialization;
    at[0].val.programmaticStreamSerializationAllowed = 1;
    cfg.attrs = at;
    cfg.numAttrs = pdl_enabled() ? 1 : 0;
    return cudaLaunchKernelEx(&cfg, kern, std::forward<Args>(args)...);
}
#endif

// symbol variants compiled into the advection kernel
enum { SYM_LAG_D1 = 0, SYM_LAG_D4 = 1, SYM_LAG_D8 = 2, SYM_SPLINE3 = 3, SYM_COUNT = 4 };

// Per-line shift record, REC_WORDS floats, written by the shift-setup kernel (step S1):
//   [0]      b mod N as int bits                      (integer part of beta)
//   [1..9]   Lagrange: a_k(1-b*)/(2N), k=0..8         (Everett-form polynomial in s = 2-2cos(theta))
//            spline:   [1..4] = 3/(2N) * (B(b*+1), B(b*), B(b*-1), B(b*-2))
//   [10..18] Lagrange: a_k(b*)/(2N)
//   [19]     v-direction: s_i = E_i * dt (fp32) for the delta-f source; else 0
constexpr int REC_WORDS = 20;

struct AdvectArgs {
    float* f;              // [Nv][Nx]
    int Nx, Nv;
    const float2* tw;      // N roots e^{-2 pi i k/N} of the advected direction
    const float* rec;      // [n_lines][REC_WORDS]
    int lognl;             // log2(complex lines per CTA)
    int ng;                // number of Gaussians of f_eq (v-direction source), 0 = none
    const float* feq_tab;  // [ng][Nv]  amp_g exp(-c_g (v_j-mu_g)^2)
    const float* vmu_tab;  // [ng][Nv]  v_j - mu_g
    float cg[4];
};

// Per-line record of the contiguous-line (x) kernel, XREC_WORDS floats (96 B = 6 cp.async chunks):
//   [0]      b mod N as int bits (integer part of beta)
//   [1]      1/N                       (mode 0: lambda_0 = 1 exactly)
//   [2]      lambda_{N/2} / N          (Nyquist mode of the line, real)
//   [4..12]  Lagrange: a_k(1-b*)/(2N), k = 0..8;   spline: [4..7] = 3/(2N) (B(b*+1), B(b*), B(b*-1), B(b*-2))
//   [13..21] Lagrange: a_k(b*)/(2N)
constexpr int XREC_WORDS = 24;

struct AdvectXArgs {
    float* f;             // [n_lines][N], lines contiguous
    int n_groups;         // n_lines >> lpi_log
    int lpi_log;          // log2(lines per iteration)
    int nbuf;             // line buffers per CTA: 2 = prefetch the next group during the transform, 1 = none
    const float2* twA;    // [R1-1][S1]   e^{-2 pi i t q / M}
    const float2* twB;    // [15][16]     e^{-2 pi i t q / 256}
    const float2* cs;     // [N/2+1]      (cos, sin)(2 pi k / N)
    const float* rec;     // [n_lines][XREC_WORDS]
    float2 root32[32];    // e^{+2 pi i j / 32}
};

typedef cudaError_t (*advect_x_launch_fn)(const AdvectXArgs& a, int sym, int grid, int threads, size_t smem,
                                          cudaStream_t st);
advect_x_launch_fn advect_x_launcher(int N);
int advect_x_occupancy(int N, int sym, int threads, size_t smem);

// ---- overlap-save kernels (vog_os2.cuh), line length >= 1024
constexpr int OS_LB = 256;     // block length (reals)
// Kept samples V and samples discarded on the left HLO of a block (256 - V - HLO are discarded on the right):
//   Lagrange 2d+1 <= 17: the stencil reaches 8 cells to the left and 9 to the right => (232, 8), exact;
//   cubic spline: the circulant row decays like 0.268^|j|; cut 14 cells either side => (228, 14): the
//   neglected part of the row sums to <= 8.4e-9 of max|u| over all b* (reading Q6b), 0.4 % of the tolerance.
constexpr int OS_V = 228;      // spline geometry: kept samples per block
constexpr int OS_H = 14;       // spline geometry: discarded on the left (and on the right)
constexpr int OS_VL = 232;     // Lagrange geometry
constexpr int OS_HL = 8;
// Per-line symbol table, OS_LAMW float2 (1040 B): [k] = lambda(2 pi k/OS_LB) / OS_LB, k = 0..128;
// [129] = (integer shift b mod N as int bits;  v: s = E dt of the delta-f source).
constexpr int OS_LAMW = 130;

struct OsArgs {
    const float* src;      // [Nv][Nx]
    float* dst;            // x: may equal src; v: must differ
    int Nx, Nv;
    int N;                 // line length (x: Nx, v: Nv)
    int nb;                // blocks per line = ceil(N / V)
    const float2* lam;     // [n_lines][OS_LAMW]
    const float2* tw;      // x: [7][16] e^{-2 pi i t q/128};  v: [15][16] e^{-2 pi i t q/256}
    const float2* cs;      // [129] (cos, sin)(2 pi k/256)   (x only)
    int lpi, n_groups;     // x: lines per iteration, n_lines / lpi
    unsigned inv_nb;       // x: ceil(2^16 / nb)
    int np_log, rb, gpc;   // v: log2(column pairs per strip), row blocks per group, groups per CTA
    int ng;                // v: Gaussians of f_eq (0 = no source)
    const float* feq_tab;  // [ng][Nv]
    const float* vmu_tab;  // [ng][Nv]
    float cg[4];
    const float* cg4;      // the same four constants in device memory (dynamic indexing)
    float dvf;             // v: dv as float (row stride of the delta-f source recurrence)
    int np;                // second-generation kernels (vog_os2.cuh): pairs of blocks per line = ceil(nb / 2)
    unsigned inv_np;       // x: ceil(2^16 / np)
    int n_lines;           // x: number of lines (the last line group may be ragged)
    int lam_ks;            // v: row stride of the transposed symbol table [k][column] in float2 (Nx + 16)
    int inplace;           // v (osv7_kernel): dst == src, whole strips per CTA, stored in place where the shifts allow it
    float* dst2;           // ... second grid for the strips whose shifts do not
    int* strip_flags;      // ... [Nx / 16] 1 = the strip went to dst2 (cleared by the copy-back kernel)
    float* halo;           // ... [CTAs][4][2][40][16] rows on either side of the pieces that are not whole strips
};

struct OsSetupArgs {
    int n_lines, N, mode;      // mode 0: c = v_l; 1: c = E_l (+E_ext_l); 2: explicit beta
    int spline, d, vdir;
    int ks;                    // vdir: row stride of the transposed table [k][line] in float2
    double dt, delta, vmin, dv;
    const float* E;
    const float* Eext;
    const double* beta;
    const double2* cs64;       // [OS_LB] (cos, sin)(2 pi j / OS_LB) in fp64
    float2* lam;
    // field solve fused into the v kernel (osv7_kernel, one piece per CTA; vog_lib.cu field_then_v): fpart != NULL => E
    // is not read but COMPUTED from the density kernel's slab sums as the circular convolution of rho with the Green's
    // function of the Fourier solve (green: [N lines] doubles), and written to E_out / rho_out by the strip's first CTA
    const double* fpart;       // [n_lines] rho of the density kernel (its last blocks add the slabs; NULL: E is given)
    const double* green;       // [n_lines]
    int nby;
    float* E_out;              // [n_lines] self-consistent field (without E_ext)
    double* rho_out;           // [n_lines]
    double* energy_out;        // (1/2) dx sum E^2 of this field solve, or NULL
    double* e_part;            // [n_lines / 16] per-strip sums of E^2 (scratch of the energy reduction)
    unsigned* ticket;          // arrival counter of the energy reduction (zero between launches)
    double half_dx;
    int spec;                  // osv7_kernel: request every group's first window before the field is known (shifts < 16 rows)
};

cudaError_t os_setup_launch(const OsSetupArgs& s, cudaStream_t st);
// per-device cudaFuncAttributeMaxDynamicSharedMemorySize (vog_os.cu)
cudaError_t set_max_smem(const void* fn, size_t smem);
cudaError_t osx7_launch(const OsArgs& a, int geom, int grid, int threads, size_t smem, cudaStream_t st);
int osx7_occupancy(int geom, int threads, size_t smem);
cudaError_t osx6_launch(const OsArgs& a, int geom, int grid, int threads, size_t smem, cudaStream_t st);
int osx6_occupancy(int geom, int threads, size_t smem);
cudaError_t osv7_launch(const OsArgs& a, const OsSetupArgs& su, int geom, int n_sm, cudaStream_t st);
cudaError_t strip_copy_launch(float* dst, const float* src, int* strip_flags, int Nx, int Nv, cudaStream_t st);
cudaError_t osv6_launch(const OsArgs& a, int geom, dim3 grid, cudaStream_t st);
cudaError_t osv4_launch(const OsArgs& a, int geom, dim3 grid, int threads, size_t smem, cudaStream_t st);

// ---- direct-stencil kernels (vog_stencil.cu): the same circulant product without the transforms (NEXT-4)
cudaError_t st_setup_launch(const OsSetupArgs& s, float* taps, cudaStream_t st);
size_t stx_smem_bytes(int spline, int d, int threads);
cudaError_t stx_launch(const OsArgs& a, int spline, int d, const float* taps, int grid, int threads, size_t smem, cudaStream_t st);
int stx_occupancy(int spline, int d, int threads, size_t smem);
cudaError_t stv_launch(const OsArgs& a, int spline, int d, const float* taps, cudaStream_t st);

// ---- one persistent kernel for a whole run of a small grid (vog_small.cu, NEXT-1; Nx, Nv <= 256)
struct SmallArgs {
    float* f;                  // [Nv][Nx], in place
    float* E_out;              // [Nx] self-consistent field of the last field solve (or NULL)
    const float* E_init;       // VXV: field for the first half step (NULL: solved from f first)
    const float* E_ext_seq;    // [n_vadv][Nx] or NULL
    double* energy;            // [n_field] or NULL
    int Nx, Nv, rpc;           // rpc = rows per CTA = Nv / cluster size
    int split, merge, nsteps, spline, d, ng;
    double dt, L, vmin, dv, dx;
    double amp[4], mu[4], c[4];
    float cg[4];
};
int small_run_cluster(int Nx, int Nv);
cudaError_t small_run_launch(const SmallArgs& a, cudaStream_t st);

// ---- double-precision mode (vog_f64.cu, NEXT-2): its own tables and kernels, created on the first *_f64 call of a plan
struct F64State;
int f64_create(F64State** out, const vog_params_t* p, cudaStream_t st, int n_sm);
void f64_destroy(F64State* S);
long long f64_launches(const F64State* S);
bool f64_has_field(const F64State* S);
cudaError_t f64_shift(F64State* S, double* f, const double* beta, bool vdir);
cudaError_t f64_advect_x(F64State* S, double* f, double dt);
cudaError_t f64_advect_v(F64State* S, double* f, const double* E, double dt);
cudaError_t f64_field(F64State* S, const double* f, double* E_out);
cudaError_t f64_get_field(F64State* S, double* E);
cudaError_t f64_step(F64State* S, double* f, double dt, const double* Eext);

// launchers, one family per line length N (defined in vog_advect_inst.cu, compiled once per N)
typedef cudaError_t (*advect_launch_fn)(const AdvectArgs& a, int sym, bool vdir, int n_tiles, int threads,
                                        size_t smem, cudaStream_t st);
advect_launch_fn advect_launcher(int N);
size_t advect_smem_bytes(int N, int lognl);

#define VOG_DECL_LAUNCH(NN) cudaError_t advect_launch_##NN(const AdvectArgs&, int, bool, int, int, size_t, cudaStream_t); \
    cudaError_t advect_x_launch_##NN(const AdvectXArgs&, int, int, int, size_t, cudaStream_t); \
    int advect_x_occ_##NN(int, int, size_t);
// whole-line kernels serve line lengths <= 512; longer lines use the overlap-save kernels
VOG_DECL_LAUNCH(64) VOG_DECL_LAUNCH(128) VOG_DECL_LAUNCH(256) VOG_DECL_LAUNCH(512)
#undef VOG_DECL_LAUNCH

}  // namespace vog
