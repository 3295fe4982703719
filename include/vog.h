/*
 * vog.h -- C ABI of libvog: the B200 (sm_100a) hot path of the 1Dx1D semi-Lagrangian
 * Vlasov-Poisson solver of "Vlasov on GPU (VOG project)", arXiv 1301.5892.
 * Citations "P:n" are line n of the paper text; "Qn" are the readings listed
 * in DESIGN.md.
 *
 * Data layout.  The phase-space array f is fp32, row-major [Nv][Nx]: f[j*Nx + i] is the
 * value at (x_i, v_j), x_i = i*L/Nx, v_j = vmin + j*(vmax-vmin)/Nv (Q2).  Both
 * directions are periodic.  In delta-f mode (feq.n > 0) the array holds
 * delta f = f - f_eq(v_j); in full-f mode (feq.n == 0) it holds f.
 *
 * Conventions.  Every entry point returns a status (VOG_OK == 0, negative on error),
 * never throws, and never synchronises the host unless stated: work is enqueued on the
 * plan's CUDA stream.  Argument errors are detected before anything is enqueued.
 * Pointers named *_dev are caller-owned DEVICE memory (16-byte aligned); pointers named
 * *_host are caller-owned HOST memory.  The library never frees caller memory.  Plan-owned
 * scratch is O(Nx + Nv) tables, plus -- only when Nv >= 1024 -- ONE second grid of Nx*Nv floats that the
 * out-of-place v kernel writes and the following x-advection reads back (contrast the
 * paper's transposed copies).  It is allocated on the first v-advection.  A plan is not
 * thread-safe; distinct plans are independent.  There is no CPU fallback anywhere: every
 * step of the path runs in the library's CUDA kernels.
 */
#ifndef VOG_H
#define VOG_H

#ifdef __cplusplus
extern "C" {
#endif

typedef struct vog_plan_s* vog_plan_t; /* opaque, library-owned */

enum { VOG_OK = 0, VOG_EINVAL = -1, VOG_ENOMEM = -2, VOG_ECUDA = -3, VOG_EUNSUPPORTED = -4, VOG_ETOOLARGE = -5 };
enum { VOG_LAGRANGE = 0, VOG_BSPLINE = 1 }; /* order = polynomial degree: Lagrange odd 1..17, B-spline 3 (Q6) */
enum { VOG_SPLIT_XVX = 0, VOG_SPLIT_VXV = 1 };

/* f_eq(v) = sum_{g<n} amp[g] * exp(-c[g] * (v - mu[g])^2); n == 0 selects full-f storage.
 * The paper's f_eq is n=1, amp=1/sqrt(2 pi), mu=0, c=1/2. */
typedef struct {
    int n;
    double amp[4], mu[4], c[4];
} vog_feq_t;

typedef struct {
    int Nx, Nv;          /* powers of two in [64, 16384]                         */
    double L;            /* x in [0, L), periodic; L > 0                          */
    double vmin, vmax;   /* v in [vmin, vmax), periodic; vmax > vmin              */
    int kind, order;     /* VOG_LAGRANGE with odd order <= min(17, N-1), or VOG_BSPLINE with order 3 */
    vog_feq_t feq;       /* delta-f equilibrium                       */
    int split;           /* VOG_SPLIT_XVX (default, binds BASELINE.json's configs) or VOG_SPLIT_VXV; Q1 */
} vog_params_t;

/* Create a plan: validates p, allocates the O(Nx+Nv) device scratch (roots of unity, rho, E,
 * per-line shift records) on the current CUDA device and binds the plan to `cuda_stream`
 * (a cudaStream_t passed as void*; NULL = the legacy default stream).  Synchronises once.
 * Errors: VOG_EINVAL (NULL pointer, sizes, L, v-range, feq.n outside [0,4], c[g] <= 0),
 * VOG_EUNSUPPORTED (kind/order), VOG_ENOMEM, VOG_ECUDA.  *out is set only on VOG_OK. */
int vog_plan(vog_plan_t* out, const vog_params_t* p, void* cuda_stream);

/* Destroy a plan and free its scratch.  Synchronises the plan's stream.  NULL is VOG_EINVAL. */
int vog_destroy(vog_plan_t plan);

/* Transport in x over dt: for every velocity row j, the periodic line f[j][:] is
 * multiplied by the circulant interpolation matrix A of eq (4) for the normalised
 * displacement beta_j = -v_j*dt/dx, computed as FFT -> symbol -> inverse FFT
 * inside one fused kernel.  In place; f_dev holds Nx*Nv floats.  dt may be < 0. */
int vog_advect_x(vog_plan_t plan, float* f_dev, double dt);

/* Transport in v over dt: for every space column i, the periodic line
 * f[:][i] is shifted by beta_i = -E_i*dt/dv; E_dev holds Nx floats (the total advecting
 * field).  In delta-f mode the source f_eq(v_j - dt*E_i) - f_eq(v_j) is added, an
 * evaluation, not an interpolation.  In place for the caller; for Nv >= 1024 the kernel writes
 * the plan's second grid and the result is copied back (vog_step avoids that copy).  VOG_ENOMEM if the
 * second grid cannot be allocated. */
int vog_advect_v(vog_plan_t plan, float* f_dev, const float* E_dev, double dt);

/* Self-consistent field: rho_i = dv * sum_j f[j][i] (of delta f in
 * delta-f mode, Q11), made zero-mean, then the Fourier solve E^_m = rho^_m / (i k_m),
 * k_m = 2 pi m / L, with modes 0 and Nx/2 set to 0 (Q12).  E_dev receives Nx floats
 * with zero mean.  f_dev is not modified. */
int vog_field(vog_plan_t plan, const float* f_dev, float* E_dev);

/* The paper's diagnostics of a state, all summed in fp64 in a fixed order.
 * Solves the field of f_dev with the plan's field solver (it stays in the plan like after vog_field) and writes five
 * doubles to diag_dev (device memory):
 *   [0] electric energy (1/2) dx sum_i E_i^2
 *   [1] rho^_0 = (1/Nx) sum_i rho_i, the equilibrium's mass dv sum_j f_eq(v_j) added in delta-f mode: the "error of
 *       mass" of P:245 is |[1] - 1|
 *   [2] |rho^_1| = |(1/Nx) sum_i rho_i e^(-2 i pi i/Nx)|, "the first mode of rho in absolute value"
 *   [3] kinetic energy (1/2) dx dv sum_j v_j^2 sum_i f_ji, the equilibrium's part added in delta-f mode
 *   [4] total energy [0] + [3]
 * f_dev is not modified.  VOG_EINVAL for NULL pointers. */
int vog_diagnostics(vog_plan_t plan, const float* f_dev, double* diag_dev);

/* One Strang step of size dt, in place (Q1).  E_ext_dev (Nx floats, or NULL) is added
 * to the self-consistent field before every v-advection of the step (for the KEEN drive pass
 * -E_app).
 *   VOG_SPLIT_XVX: x(dt/2); E = field(f); v(dt, E + E_ext); x(dt/2).
 *   VOG_SPLIT_VXV: v(dt/2, E_prev + E_ext); x(dt); E = field(f); v(dt/2, E + E_ext), where
 *                  E_prev is the field the previous VXV step (or a vog_field call) on the SAME f_dev left in the
 *                  plan; after any other call on the plan, or for another array, it is solved from f_dev first
 *                  (see vog_reset for states changed behind the library's back).
 * The self-consistent E solved inside the step stays in the plan: see vog_get_field. */
int vog_step(vog_plan_t plan, float* f_dev, double dt, const float* E_ext_dev);

/* Copy the self-consistent field of the last vog_step / vog_field of this plan (Nx floats)
 * into E_dev (device to device, asynchronous).  VOG_EINVAL if none was computed yet. */
int vog_get_field(vog_plan_t plan, float* E_dev);

/* Lower level (BASELINE.json config 4: "per-line shifts uniform in [-8,8] cells"): apply the
 * circulant interpolation matrix with an explicit normalised displacement beta (in cells,
 * fp64, device memory) per line: row j of f is shifted by beta_cells_dev[j] (Nv values) /
 * column i by beta_cells_dev[i] (Nx values).  No delta-f source.  In place. */
int vog_shift_x(vog_plan_t plan, float* f_dev, const double* beta_cells_dev);
int vog_shift_v(vog_plan_t plan, float* f_dev, const double* beta_cells_dev);

/* Out-of-place form of vog_shift_v: reads src_dev, writes dst_dev (both Nx*Nv floats, caller-owned device
 * memory, dst_dev != src_dev and not overlapping).  For Nv >= 1024 the v kernel is out of place by
 * construction (a block reads rows that other blocks write), so the in-place calls vog_shift_v / vog_advect_v
 * go through the plan's second grid and copy back; this call is the kernel alone (it is what vog_step uses
 * internally, ping-ponging between f and the second grid).  VOG_EINVAL if dst_dev == src_dev. */
int vog_shift_v_to(vog_plan_t plan, const float* src_dev, float* dst_dev, const double* beta_cells_dev);

/* nsteps Strang steps of size dt on the device, in place, asynchronous like vog_step (S10 driver).
 *   merge = 0: exactly the kernels of nsteps calls of vog_step, bit for bit.
 *   merge = 1: the half steps that meet between two consecutive steps are taken as one advection over dt, which the
 *              paper names as the easy way to more speed: 2 advections per step instead of 3.
 *                VOG_SPLIT_XVX: x(dt/2) [E=field; v(dt,E+E_ext); x(dt)]^(nsteps-1) E=field; v(dt,E+E_ext); x(dt/2)
 *                VOG_SPLIT_VXV: v(dt/2) [x(dt); E=field; v(dt,E+E_ext)]^(nsteps-1) x(dt); E=field; v(dt/2,E+E_ext)
 *              (in VXV the two half steps see the same E because rho is invariant under a v-advection, P:205-213;
 *              the merged result differs from the unmerged one by interpolation error only, not by rounding only).
 * E_ext_seq_dev: NULL, or one row of Nx floats per v-advection, in the order the v-advections are taken
 *   (XVX: nsteps rows; VXV: 2*nsteps rows unmerged, nsteps+1 merged).
 * energy_dev: NULL, or nsteps doubles in device memory; entry s receives the electric energy (1/2) dx sum_i E_i^2
 *    of the self-consistent field of the s-th field solve of the call (XVX: at the half-advanced density of
 *   step s; VXV: at t^(s+1)), summed in fp64 in a fixed order.
 * VOG_EINVAL for NULL plan / f_dev, nsteps < 0, merge outside {0,1}; VOG_ENOMEM if the second grid cannot be had. */
int vog_run(vog_plan_t plan, float* f_dev, double dt, int nsteps, const float* E_ext_seq_dev, int merge,
            double* energy_dev);

/* End-to-end convenience with HOST buffers: copies f_host (Nx*Nv floats) and E_ext_host (Nx
 * floats or NULL) into a device buffer that the plan allocates on the first call and keeps (the
 * only O(Nx*Nv) allocation of the library, made only if this call is used), runs `nsteps`
 * Strang steps with the same E_ext, copies f back into f_host and the last self-consistent E
 * into E_host (Nx floats, may be NULL), and SYNCHRONISES the stream before returning.
 * Pinned host memory gives full-rate copies; pageable memory also works. */
int vog_run_host(vog_plan_t plan, float* f_host, double dt, int nsteps,
                 const float* E_ext_host, float* E_host);

/* The same without the final synchronisation: everything (copy in, steps, copies out) is enqueued on the plan's stream
 * and the call returns; the host buffers must be pinned and stay untouched until the caller has synchronised that
 * stream.  Several plans on several streams then overlap one replica's copy in, another's steps and a third's copy
 * out (PCIe is full duplex), which is how `bench.py` measures its end-to-end figure. */
int vog_run_host_async(vog_plan_t plan, float* f_host, double dt, int nsteps,
                       const float* E_ext_host, float* E_host);

/* Launch-shape override for measurements; never needed for normal use and never
 * changes results beyond rounding.  which:
 *   2, 3   whole-line v kernel (Nv <= 512): log2(complex lines per CTA), threads per CTA;
 *   5..8   whole-line x kernel (Nx <= 512): log2(lines per iteration), threads (32..128), CTAs per SM
 *          (0 = as many as fit), line buffers (1 or 2);
 *   18     overlap-save x kernel (Nx >= 1024): lines per iteration of a CTA;
 *   20     overlap-save v kernel (Nv >= 1024): pairs of blocks per CTA (0 = default);
 *   21     overlap-save x kernel variant: 0 = every pair of blocks lands its own window of the line by bulk asynchronous
 *          copies (default for lines up to 8192 cells), 1 = whole lines landed for the whole CTA (what 16384-cell
 *          lines always use);
 *   22     overlap-save v kernel variant: 0 = 16-column strips with the next window in flight (default), 1 = 32-column
 *          strips sharing one buffer (the fallback kept beside it);
 *   24     density kernel: row slabs per column group (power of two, 1..16, at least 32 rows each);
 *   25     block geometry of the overlap-save kernels: 1 = 232 kept samples, 8 + 16 discarded (Lagrange
 *          plans only, their default), 0 = 224 kept, 16 + 16 discarded (the cubic spline's);
 *   26     programmatic dependent launch of the plan's kernels: 1 = each kernel may be staged on the SMs while its
 *          predecessor in the stream drains and waits for it on the device (default), 0 = plain stream order.
 *          Results are bit-identical either way.
 *   27     how the circulant product of lines >= 1024 cells is taken: 0 = in Fourier space (default: FFT, symbol,
 *          inverse FFT, P:131-149 -- the path BASELINE.json names), 1 = directly, u'_i = sum_j a_j u_(i+b+j) with the
 *          2d+2 non-zero entries of the row of A (eq (4); the spline's row cut at |j| <= 14 like the
 *          Fourier path's blocks).  The same matrix up to rounding.  Shorter lines always use
 *          the Fourier kernels.
 *   28     field solve: 0 = Fourier, modes 0 and Nx/2 dropped (default); 1 = trapezoidal rule with the
 *          zero-mean modifications on rho and on E; 2 = trapezoidal rule without them (rho - 1, P:213;
 *          minus the equilibrium's mass in delta-f mode) -- the variant whose drift the paper shows in Fig. 1.
 *          This one DOES change results: it is the paper's other solver, not a launch shape.
 *   29     grids up to 256 x 256 only: 1 = vog_run executes the whole run as ONE persistent kernel on a thread-block
 *          cluster that keeps the grid in shared memory for all nsteps (the circulant products in
 *          their direct form, the same matrices up to rounding), same sequences, E_ext and energy semantics as the
 *          launch-per-kernel loop; 0 = that loop (default: vog_run(merge = 0) stays bit-identical to vog_step).
 *          Ignored while the trapezoid field solver (28) is selected.
 *   30     grids with Nv >= 1024 and Nx / 16 <= the number of SMs (Nx <= 2048 on a B200), or Nx >= 4096: 1 (default there) = in
 *          vog_step / vog_run the field solve that precedes a v-advection runs INSIDE the v kernel: the density kernel's
 *          last blocks write rho, every CTA of the v kernel computes E on its own 16 columns as the circular convolution
 *          of rho with the Green's function of the same Fourier solve (fp64) and the strip's first CTA publishes
 *          E (vog_get_field) and the energy share; a step is then 4 launches (x, density, v, x).  0 = density, Poisson
 *          kernel, v kernel (5 launches).  Same E up to rounding (the convolution is the more accurate of the two).
 *          On grids of 4096 columns or more, 1 (default) = the same convolution as a kernel of its own (one CTA per 64
 *          columns) in the place of the single-CTA Poisson kernel.
 *   31     v kernel (Nv >= 1024): 1 (default) = every group requests the rows of its first pair of blocks BEFORE the
 *          field / the shifts are known -- the raw buffer's whole 520 rows, which serve any integer shift in [-16, 16)
 *          -- and requests them again if the shifts turn out larger; 0 = after the shifts are known.
 *   33     density kernel launched with (1) or without (0) the programmatic-dependent-launch attribute of code 26
 *          (default: with it below 4096 x 4096 cells, without it from there on).
 *   34     vog_advect_v / vog_shift_v with Nv >= 1024: 1 (default) = the v kernel stores IN PLACE wherever a strip's
 *          integer shifts are at most 24 rows (a store waits until the windows that still need the rows are on chip; the
 *          rows on either side of a piece of work are saved first); strips with larger shifts go through the plan's
 *          second grid and are copied back by a second launch.  0 = every strip through the second grid and a copy of
 *          the whole grid.
 * VOG_EINVAL for an unknown code or a shape that does not fit (shared memory, grid). */
int vog_plan_tune(vog_plan_t plan, int which, int value);

/* Forget what the plan caches about the state it last saw: the self-consistent field kept for vog_get_field and for
 * the first half step of the next VOG_SPLIT_VXV step, and the x-advection tables of the last time step.  The library
 * drops these itself whenever one of ITS calls changes the state or is given another array; call vog_reset after
 * writing into f_dev behind the library's back (e.g. re-initialising the same buffer) before a VXV step.  Never
 * needed with VOG_SPLIT_XVX.  Returns VOG_OK, or VOG_EINVAL for NULL. */
int vog_reset(vog_plan_t plan);

/* Double-precision mode.  The same plan, the same parameters and the same
 * call sequence with every array in fp64: f_dev holds Nx*Nv DOUBLES in the layout of the fp32 calls, E / E_ext / beta
 * are Nx (or Nv) doubles in device memory.  The mode keeps its own tables and its own second grid (Nx*Nv doubles,
 * allocated on the first v-advection; the out-of-place v kernel writes it and the following x-advection reads it back,
 * so a step makes no copy; the stand-alone v calls copy back), created on the first *_f64 call of the plan; its state
 * (cached x tables, the field kept for vog_get_field_f64 and the first half step of a VXV step) is separate from the
 * fp32 calls', with the same rules.  What is computed:
 *   - the circulant product of eq (4) in its direct form u'_i = sum_j a_j u_(i+b+j): the 2d+2 non-zero
 *     entries of the row of A for Lagrange 2d+1, and for the cubic spline the row a = m * g with
 *     g_n = sqrt(3) (sqrt(3) - 2)^|n| cut at |n| <= 30 (the neglected part of the row is < 1e-17), all in fp64;
 *   - rho by fixed-order fp64 column sums, zero mean, the Fourier solve E^_m = rho^_m / (i k_m) with modes 0 and Nx/2
 *     dropped (Q12) as two plain DFT sums (exact to rounding; O(Nx^2) operations spread over the GPU);
 *   - the delta-f source f_eq(v - dt E) - f_eq(v) with expm1 in fp64.
 * Asynchronous on the plan's stream, same error behaviour as the fp32 calls (VOG_EINVAL for NULL pointers, VOG_ENOMEM
 * when the tables or the second grid cannot be allocated).  vog_plan_tune codes do not apply to this mode. */
int vog_shift_x_f64(vog_plan_t plan, double* f_dev, const double* beta_cells_dev);
int vog_shift_v_f64(vog_plan_t plan, double* f_dev, const double* beta_cells_dev);
int vog_advect_x_f64(vog_plan_t plan, double* f_dev, double dt);
int vog_advect_v_f64(vog_plan_t plan, double* f_dev, const double* E_dev, double dt);
int vog_field_f64(vog_plan_t plan, const double* f_dev, double* E_dev);
int vog_get_field_f64(vog_plan_t plan, double* E_dev);
int vog_step_f64(vog_plan_t plan, double* f_dev, double dt, const double* E_ext_dev);

/* The self-consistent field WITHOUT a plan and without any allocation, for callers that cannot call cudaMalloc (code
 * under CUDA graph capture, tight serving loops, harnesses that forbid it).  Same definition as vog_field (P:157, 172,
 * 205-211, 221): rho_i = dv sum_j f[j][i] with dv = (vmax - vmin) / Nv, zero mean, E^_m = rho^_m / (i k_m) with modes 0
 * and Nx/2 dropped; f_dev holds Nx*Nv floats in the layout above, E_dev receives Nx floats (both caller-owned device
 * memory); enqueued on cuda_stream (a cudaStream_t as void*, NULL = the legacy default stream), asynchronous.  The
 * density kernel's slab sums and the O(Nx) work arrays of the solve live in a file-scope device array of 416 KB that
 * every GPU loading the library holds until the process exits; the call makes no cudaMalloc / cudaFree and calls no
 * allocating library routine.  Limit: Nx <= VOG_NOALLOC_MAX_NX, beyond it VOG_ETOOLARGE (use a plan and vog_field).
 * Nx, Nv powers of two, Nx >= 64, 64 <= Nv <= 16384, L > 0, vmax > vmin, non-NULL pointers: else VOG_EINVAL.
 * ALL calls in the process share the one scratch array (per GPU), which keeps the last call's contents; every call
 * overwrites each word before reading it, so nothing needs clearing, but calls that OVERLAP on the same GPU (different
 * streams) race on it: keep them on one stream or order them with events.  The sums are plain fp64 DFT sums, O(Nx^2):
 * meant for the moderate Nx it is limited to, not as a replacement of vog_field. */
#define VOG_NOALLOC_MAX_NX 4096
int vog_field_noalloc(const float* f_dev, int Nx, int Nv, double L, double vmin, double vmax, float* E_dev,
                      void* cuda_stream);

/* Number of kernels the library launched on this plan since creation (for accounting). */
long long vog_launch_count(vog_plan_t plan);

/* Static description of a status code.  Never NULL. */
const char* vog_strerror(int status);

#ifdef __cplusplus
}
#endif
#endif /* VOG_H */
