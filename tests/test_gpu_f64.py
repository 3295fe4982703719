"""GPU parity of the double-precision mode (include/vog.h "*_f64"): the CUDA path through the
C ABI against the fp64 oracle, element by element on the same seeded inputs.  Run with `-m gpu` on the B200 box.

Tolerances, relative to max|input|: one advection is a sum of at most 64 products with
sum_j |a_j| <= 3.3 (Lagrange 17), so 64 * 2^-53 * 3.3 ~ 2.4e-14 bounds its rounding and 2e-13 is asked for; the
field is a sum of Nv terms followed by two sums of Nx terms: 1e-11 of max|E| is asked for up to 2048 points; a
step is three advections and a field solve: 1e-11 of max|f|.  Fifty million times tighter than the fp32 path's 2e-6.
"""
import math

import numpy as np
import pytest

from paper_1301_5892_b200 import inputs

pytestmark = pytest.mark.gpu

LAG, SPL = 0, 1
ALL_KINDS = [(LAG, 1), (LAG, 3), (LAG, 5), (LAG, 9), (LAG, 13), (LAG, 17), (SPL, 3)]


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
    return torch.from_numpy(np.ascontiguousarray(a, dtype=np.float64)).cuda()


def _shifts(n, seed):
    beta = inputs.uniform_shifts(n, seed)
    special = [0.0, 3.0, -5.0, -0.25, 0.999999, 1e-9, -1e-9, 123456.75, -98765.5, 7.5]
    beta[: len(special)] = special
    return beta


def _rel(out, ref, scale):
    return float(np.abs(out - ref).max() / scale)


@pytest.mark.parametrize("kind,order", ALL_KINDS)
@pytest.mark.parametrize("Nx,Nv", [(64, 64), (128, 256), (1024, 128), (256, 2048), (2048, 512)])
def test_f64_shift_parity_both_directions(torch, vog, oracle, Nx, Nv, kind, order):
    rng = np.random.default_rng(5 + Nx + Nv)
    f = rng.random((Nv, Nx))                                  # full fp64 mantissas (not fp32 values promoted)
    plan = vog.Plan(Nx, Nv, 4 * math.pi, -6.0, 6.0, kind, order)
    bx, bv = _shifts(Nv, 11), _shifts(Nx, 12)
    fd = _dev(torch, f)
    plan.shift_x_f64(fd, _dev(torch, bx))
    torch.cuda.synchronize()
    assert _rel(fd.cpu().numpy(), oracle.shift_x(f, bx, kind, order), np.abs(f).max()) <= 2e-13
    fd = _dev(torch, f)
    plan.shift_v_f64(fd, _dev(torch, bv))
    torch.cuda.synchronize()
    assert _rel(fd.cpu().numpy(), oracle.shift_v(f, bv, kind, order), np.abs(f).max()) <= 2e-13
    plan.destroy()


def test_f64_shift_is_really_double(torch, vog, oracle):
    """The same shift through the fp32 calls differs from the oracle by ~1e-7: the fp64 mode must not be the fp32
    kernels behind a conversion."""
    Nx = Nv = 1024
    rng = np.random.default_rng(9)
    f = rng.random((Nv, Nx))
    bx = _shifts(Nv, 3)
    plan = vog.Plan(Nx, Nv, 1.0, -1.0, 1.0, LAG, 17)
    f32 = torch.from_numpy(f.astype(np.float32)).cuda()
    plan.shift_x(f32, _dev(torch, bx))
    f64 = _dev(torch, f)
    plan.shift_x_f64(f64, _dev(torch, bx))
    torch.cuda.synchronize()
    ref = oracle.shift_x(f, bx, LAG, 17)
    e32 = np.abs(f32.cpu().numpy().astype(np.float64) - ref).max()
    e64 = np.abs(f64.cpu().numpy() - ref).max()
    assert e64 <= 2e-13 and e32 >= 1e-9 and e32 <= 2e-6
    plan.destroy()


@pytest.mark.parametrize("idx", [0, 1, 2])
def test_f64_field_parity(torch, vog, oracle, idx):
    cfg = inputs.config(idx)
    f = inputs.initial_f(cfg).astype(np.float64)
    plan = vog.Plan.from_config(cfg)
    fd = _dev(torch, f)
    Ed = torch.empty(cfg.Nx, device="cuda", dtype=torch.float64)
    plan.field_f64(fd, Ed)
    E2 = torch.empty_like(Ed)
    plan.get_field_f64(E2)
    torch.cuda.synchronize()
    Eo = oracle.field(f, cfg.L, cfg.vmin, cfg.vmax)
    assert _rel(Ed.cpu().numpy(), Eo, np.abs(Eo).max()) <= 1e-11
    assert np.array_equal(Ed.cpu().numpy(), E2.cpu().numpy())
    assert abs(float(Ed.sum())) <= 1e-12 * cfg.Nx * float(Ed.abs().max())        # zero mean
    assert np.array_equal(fd.cpu().numpy(), f)                                     # f is not modified
    plan.destroy()


@pytest.mark.parametrize("kind,order", [(LAG, 3), (LAG, 17), (SPL, 3)])
def test_f64_advect_with_deltaf_source(torch, vog, oracle, kind, order):
    """vog_advect_x_f64 / vog_advect_v_f64 against the oracle, two off-centre Gaussians as f_eq (the source of P:197)."""
    cfg = inputs.config(2, Nx=256, Nv=512, kind=kind, order=order)
    f = inputs.initial_f(cfg).astype(np.float64)
    rng = np.random.default_rng(4)
    E = 0.3 * rng.standard_normal(cfg.Nx)
    plan = vog.Plan.from_config(cfg)
    fd = _dev(torch, f)
    plan.advect_v_f64(fd, _dev(torch, E), 0.37)
    torch.cuda.synchronize()
    ref = oracle.advect_v(f, E, cfg.vmin, cfg.vmax, 0.37, kind, order, oracle.Feq.make(cfg.feq))
    scale = max(np.abs(f).max(), np.abs(ref).max())
    assert _rel(fd.cpu().numpy(), ref, scale) <= 2e-13
    fd = _dev(torch, f)
    plan.advect_x_f64(fd, -0.21)
    torch.cuda.synchronize()
    assert _rel(fd.cpu().numpy(), oracle.advect_x(f, cfg.L, cfg.vmin, cfg.vmax, -0.21, kind, order), np.abs(f).max()) <= 2e-13
    plan.destroy()


@pytest.mark.parametrize("split", [0, 1])
@pytest.mark.parametrize("idx,over", [(0, {}), (1, {}), (2, {"Nx": 512, "Nv": 1024}), (3, {"Nx": 1024, "Nv": 256})])
def test_f64_step_parity(torch, vog, oracle, idx, over, split):
    """Three consecutive steps with an external field against the oracle's; VXV reuses the field of the previous step
    (the oracle is handed E_in the same way)."""
    cfg = inputs.config(idx, split=split, **over)
    f = inputs.initial_f(cfg).astype(np.float64)
    feq = oracle.Feq.make(cfg.feq)
    plan = vog.Plan.from_config(cfg)
    fd = _dev(torch, f)
    Ed = torch.empty(cfg.Nx, device="cuda", dtype=torch.float64)
    fo, E_in = f, None
    for n in range(3):
        ext = 0.05 * np.cos(2 * np.pi * (np.arange(cfg.Nx) / cfg.Nx) - 0.3 * n)
        plan.step_f64(fd, cfg.dt, _dev(torch, ext))
        plan.get_field_f64(Ed)
        torch.cuda.synchronize()
        fo, Eo = oracle.step(fo, cfg.L, cfg.vmin, cfg.vmax, cfg.dt, cfg.kind, cfg.order, feq, split, E_ext=ext, E_in=E_in)
        E_in = Eo if split == 1 else None
        assert _rel(fd.cpu().numpy(), fo, max(np.abs(f).max(), 1e-3)) <= 1e-11
        # (config 3 starts from delta f = 0: its first self-consistent field is exactly zero, the drive sets the scale)
        assert _rel(Ed.cpu().numpy(), Eo, max(np.abs(Eo).max(), np.abs(ext).max())) <= 1e-10
    plan.destroy()


def test_f64_long_run_follows_the_oracle_where_fp32_cannot(torch, vog, oracle):
    """what double precision buys.  40 steps of config 0 (linear Landau damping, 64 x 64): the fp64 mode
    stays within 1e-10 of the oracle's state, the fp32 path within its own 1e-4 but no better than 1e-8."""
    cfg = inputs.config(0)
    f = inputs.initial_f(cfg).astype(np.float64)
    feq = oracle.Feq.make(cfg.feq)
    plan = vog.Plan.from_config(cfg)
    f64 = _dev(torch, f)
    f32 = torch.from_numpy(f.astype(np.float32)).cuda()
    fo = f
    for _ in range(40):
        plan.step_f64(f64, cfg.dt)
        plan.step(f32, cfg.dt)
        fo, _E = oracle.step(fo, cfg.L, cfg.vmin, cfg.vmax, cfg.dt, cfg.kind, cfg.order, feq, cfg.split)
    torch.cuda.synchronize()
    scale = np.abs(f).max()
    e64 = _rel(f64.cpu().numpy(), fo, scale)
    e32 = _rel(f32.cpu().numpy().astype(np.float64), fo, scale)
    assert e64 <= 1e-10, e64
    assert 1e-8 <= e32 <= 1e-4, e32
    plan.destroy()


def test_f64_argument_errors(torch, vog):
    plan = vog.Plan(64, 64, 1.0, -1.0, 1.0, LAG, 3)
    f = torch.zeros((64, 64), device="cuda", dtype=torch.float64)
    E = torch.zeros(64, device="cuda", dtype=torch.float64)
    L = vog.lib()
    assert L.vog_get_field_f64(plan._h, vog._ptr(E)) == vog.EINVAL          # no field solved yet
    assert L.vog_step_f64(plan._h, None, 0.1, None) == vog.EINVAL
    assert L.vog_shift_x_f64(plan._h, vog._ptr(f), None) == vog.EINVAL
    assert L.vog_field_f64(None, vog._ptr(f), vog._ptr(E)) == vog.EINVAL
    assert L.vog_advect_v_f64(plan._h, vog._ptr(f), vog._ptr(E), float("nan")) == vog.EINVAL
    n0 = plan.launch_count()
    plan.step_f64(f, 0.1)
    torch.cuda.synchronize()
    assert plan.launch_count() - n0 >= 8          # 2 x (tables + x), 4 field kernels, tables + v
    plan.destroy()
