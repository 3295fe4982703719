"""GPU parity of the field solve fused into the v kernel (csrc/vog_os2.cuh osv7_kernel, csrc/vog_lib.cu field_then_v;
vog_plan_tune(30, 0/1)): on grids whose v kernel runs one piece per CTA (Nv >= 1024, Nx / 16 <= SMs) a step launches
x, density, v, x -- no Poisson kernel; every v CTA computes E on its own 16 columns as the circular convolution of rho
with the Green's function of the Fourier solve (E^_m = rho^_m / (i k_m), modes 0 and Nx/2 dropped).  On grids of
4096 columns or more the same convolution is a kernel of its own (green_field_kernel, one CTA per 64 columns) in the
single-CTA Poisson kernel's place.

Checked here: the step and its field against the oracle (same tolerances as the unfused tests), against the unfused
launch sequence, the electric energies of vog_run against the oracle's, both split orders, merged half steps,
grids with one and with several CTAs per strip, and that the fused path is really the one that ran (launch counts).
"""
import math

import numpy as np
import pytest

from paper_1301_5892_b200 import inputs

pytestmark = pytest.mark.gpu

TOL = 2e-6      # per advection, of max|f handed in| (BASELINE.json north_star)


@pytest.fixture(scope="module")
def torch():
    import torch as t
    if not t.cuda.is_available():
        pytest.skip("no CUDA device")
    return t


@pytest.fixture(scope="module")
def vog():
    from paper_1301_5892_b200 import vog as v
    v.lib()      # fails loudly if the extension is missing
    return v


def _dev(torch, a):
    return torch.from_numpy(np.ascontiguousarray(a)).cuda()


def _steps(torch, vog, cfg, f, ext, n, fuse):
    plan = vog.Plan.from_config(cfg)
    plan.tune(30, 1 if fuse else 0)
    fd = _dev(torch, f)
    ed = None if ext is None else _dev(torch, ext)
    n0 = plan.launch_count()
    for _ in range(n):
        plan.step(fd, cfg.dt, ed)
    E = torch.empty(cfg.Nx, device="cuda", dtype=torch.float32)
    launches = plan.launch_count() - n0
    plan.get_field(E)
    torch.cuda.synchronize()
    plan.destroy()
    return fd.cpu().numpy(), E.cpu().numpy(), launches


@pytest.mark.parametrize("split", [0, 1])
@pytest.mark.parametrize("idx,over", [(1, dict(Nx=1024, Nv=1024)), (2, dict(Nx=2048, Nv=1024)), (2, dict(Nx=256, Nv=2048)),
                                      (1, dict(Nx=64, Nv=4096, kind=1, order=3)), (0, dict(Nx=2048, Nv=2048)),
                                      (1, dict(Nx=4096, Nv=1024)), (2, dict(Nx=8192, Nv=256)), (1, dict(Nx=16384, Nv=128))])
def test_fused_field_step_against_oracle_and_unfused(torch, vog, oracle, idx, over, split):
    cfg = inputs.config(idx, split=split, **over)
    f = inputs.initial_f(cfg)
    ext = (0.02 * np.sin(2 * math.pi * np.arange(cfg.Nx) / cfg.Nx + 0.3)).astype(np.float32)
    n = 2
    f1, E1, l1 = _steps(torch, vog, cfg, f, ext, n, True)
    f0, E0, l0 = _steps(torch, vog, cfg, f, ext, n, False)
    # one launch fewer per fused field solve (XVX: one per step; VXV: the first step's opening solve stays unfused);
    # from 4096 columns on the x-space solve is a kernel of its own (green_field_kernel in the Poisson kernel's place)
    assert l0 - l1 == (n if cfg.Nx <= 2048 else 0)
    feq = oracle.Feq.make(cfg.feq)
    fo, Eo = f.astype(np.float64), None
    for _ in range(n):
        fo, Eo = oracle.step(fo, cfg.L, cfg.vmin, cfg.vmax, cfg.dt, cfg.kind, cfg.order, feq, split,
                             ext.astype(np.float64), Eo)
    scale = max(float(np.abs(f).max()), 1e-2 if cfg.feq else 0.0)     # (reading Q21b: delta f may start tiny)
    assert np.abs(f1 - fo).max() <= 3 * n * TOL * scale
    assert np.abs(f1.astype(np.float64) - f0).max() <= 3 * n * TOL * scale
    # (after two steps E carries the advections' rounding through rho: 1e-4 as in test_one_step_parity)
    assert np.abs(E1 - Eo).max() <= 1e-4 * np.abs(Eo).max()
    assert np.abs(E1.astype(np.float64) - E0).max() <= 2e-5 * np.abs(Eo).max()


def test_fused_field_is_the_fourier_solve(torch, vog, oracle):
    """E published by the fused step on the bench grid against oracle.field of the half-advanced state, taken from
    the GPU's own x-advection (so only the field solve differs): 2e-6 like the test of vog_field."""
    cfg = inputs.metric_config()
    f = inputs.initial_f(cfg)
    plan = vog.Plan.from_config(cfg)
    fd = _dev(torch, f)
    half = fd.clone()
    plan.advect_x(half, 0.5 * cfg.dt)
    plan.step(fd, cfg.dt)
    E = torch.empty(cfg.Nx, device="cuda", dtype=torch.float32)
    plan.get_field(E)
    torch.cuda.synchronize()
    # (delta-f: the equilibrium's density is a constant and only changes the dropped mode 0)
    Eo = oracle.field(half.cpu().numpy().astype(np.float64), cfg.L, cfg.vmin, cfg.vmax)
    assert np.abs(E.cpu().numpy() - Eo).max() <= 2e-6 * np.abs(Eo).max()
    plan.destroy()


@pytest.mark.parametrize("Nx,Nv", [(1024, 1024), (8192, 256)])
@pytest.mark.parametrize("merge", [False, True])
@pytest.mark.parametrize("split", [0, 1])
def test_fused_field_run_energies(torch, vog, oracle, split, merge, Nx, Nv):
    """vog_run with an energy per field solve: the fused reduction (strip sums added in strip order by the last strip
    to arrive; CTA sums in green_field_kernel) against the unfused kernel's and, unmerged, against the oracle's steps."""
    cfg = inputs.config(1, Nx=Nx, Nv=Nv, split=split)
    f = inputs.initial_f(cfg)
    n = 3
    outs = []
    for fuse in (1, 0):
        plan = vog.Plan.from_config(cfg)
        plan.tune(30, fuse)
        fd = _dev(torch, f)
        en = torch.zeros(n, device="cuda", dtype=torch.float64)
        plan.run(fd, cfg.dt, n, None, merge, en)
        torch.cuda.synchronize()
        outs.append((fd.cpu().numpy(), en.cpu().numpy()))
        plan.destroy()
    (f1, e1), (f0, e0) = outs
    assert np.all(e1 > 0)
    assert np.abs(e1 - e0).max() <= 1e-5 * e0.max()
    assert np.abs(f1.astype(np.float64) - f0).max() <= 3 * n * TOL * np.abs(f).max()
    if not merge:
        feq = oracle.Feq.make(cfg.feq)
        fo, Eo, eo = f.astype(np.float64), None, []
        for _ in range(n):
            fo, Eo = oracle.step(fo, cfg.L, cfg.vmin, cfg.vmax, cfg.dt, cfg.kind, cfg.order, feq, split, None, Eo)
            eo.append(oracle.electric_energy(Eo, cfg.L))
        assert np.abs(e1 - np.array(eo)).max() <= 1e-4 * max(eo)
        assert np.abs(f1 - fo).max() <= 3 * n * TOL * np.abs(f).max()


def test_fused_field_repeats_bit_for_bit_and_is_off_where_it_cannot_run(torch, vog):
    cfg = inputs.metric_config()
    f = inputs.initial_f(cfg)
    a = _steps(torch, vog, cfg, f, None, 3, True)
    b = _steps(torch, vog, cfg, f, None, 3, True)
    assert np.array_equal(a[0], b[0]) and np.array_equal(a[1], b[1])
    plan = vog.Plan(1024, 256, 1.0, -1.0, 1.0)           # whole-line v kernel, fewer than 4096 columns: no Green's function
    with pytest.raises(vog.VogError):
        plan.tune(30, 1)
    plan.destroy()


@pytest.mark.parametrize("which", [31, 33])
@pytest.mark.parametrize("idx,over", [(1, dict(Nx=2048, Nv=2048)), (2, dict(Nx=1024, Nv=2048)), (1, dict(Nx=8192, Nv=1024))])
def test_launch_shape_switches_do_not_change_a_bit(torch, vog, which, idx, over):
    """vog_plan_tune(31, .) (first windows of the v kernel requested before / after the shifts are known) and (33, .)
    (density kernel with / without the dependent-launch attribute) only change WHEN things are requested: 3 steps with an
    external field must come out bit for bit the same, field included."""
    cfg = inputs.config(idx, **over)
    f = inputs.initial_f(cfg)
    ext = (0.3 * np.cos(2 * math.pi * np.arange(cfg.Nx) / cfg.Nx)).astype(np.float32)
    outs = []
    for value in (0, 1):
        plan = vog.Plan.from_config(cfg)
        plan.tune(which, value)
        fd = _dev(torch, f)
        ed = _dev(torch, ext)
        for _ in range(3):
            plan.step(fd, cfg.dt, ed)
        E = torch.empty(cfg.Nx, device="cuda", dtype=torch.float32)
        plan.get_field(E)
        torch.cuda.synchronize()
        outs.append((fd.cpu().numpy(), E.cpu().numpy()))
        plan.destroy()
    assert np.array_equal(outs[0][0], outs[1][0]) and np.array_equal(outs[0][1], outs[1][1])


def test_speculative_window_is_redone_when_the_shifts_are_large(torch, vog, oracle):
    """A strong external field gives integer shifts far beyond the +-16 rows the speculative window covers: the v kernel
    must drop it and request the right rows (parity with the oracle's step, and the same bits as without speculation)."""
    cfg = inputs.config(1, Nx=1024, Nv=2048)
    f = inputs.initial_f(cfg)
    dv = (cfg.vmax - cfg.vmin) / cfg.Nv
    ext = (60.0 * dv / cfg.dt * np.sin(2 * math.pi * np.arange(cfg.Nx) / cfg.Nx)).astype(np.float32)   # up to 60 rows
    outs = []
    for spec in (1, 0):
        plan = vog.Plan.from_config(cfg)
        plan.tune(31, spec)
        fd = _dev(torch, f)
        plan.step(fd, cfg.dt, _dev(torch, ext))
        torch.cuda.synchronize()
        outs.append(fd.cpu().numpy())
        plan.destroy()
    assert np.array_equal(outs[0], outs[1])
    fo, _ = oracle.step(f.astype(np.float64), cfg.L, cfg.vmin, cfg.vmax, cfg.dt, cfg.kind, cfg.order,
                        oracle.Feq.make(cfg.feq), cfg.split, ext.astype(np.float64))
    # (the delta-f source of a 60-row shift is of order one: reading Q21b, the scale is that of the update)
    scale = max(float(np.abs(f).max()), float(np.abs(fo).max()))
    assert np.abs(outs[0] - fo).max() <= 3 * TOL * scale
