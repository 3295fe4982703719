"""GPU parity of the one-kernel run for small grids (vog_plan_tune(29, 1), csrc/vog_small.cu):
vog_run as ONE persistent cluster kernel against the oracle's steps and against the launch-per-kernel loop, same
sequences (both split orders, merged or not, E_ext per v-advection, energy per field solve).

Tolerance: 2e-6 of max|input| per advection (BASELINE.json north_star), i.e. (number of advections) x 2e-6 for a run;
energies at 1e-4 relative like test_run_merged_half_steps_against_oracle.
"""
import numpy as np
import pytest

from paper_1301_5892_b200 import inputs

pytestmark = pytest.mark.gpu

LAG, SPL = 0, 1
TOL = 2e-6


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


def _scale(f0, cfg):
    # (delta-f arrays can start tiny or zero: the source of P:197 sets the scale of the update, reading Q21b)
    return max(float(np.abs(f0).max()), 1e-2 if cfg.feq else 0.0)


def _run(torch, vog, cfg, f0, n, ext, merge, small):
    plan = vog.Plan.from_config(cfg)
    if small:
        plan.tune(29, 1)
    fd = _dev(torch, f0)
    en = torch.zeros(n, device="cuda", dtype=torch.float64)
    n0 = plan.launch_count()
    plan.run(fd, cfg.dt, n, None if ext is None else _dev(torch, ext), merge=merge, energy=en)
    E = torch.empty(cfg.Nx, device="cuda", dtype=torch.float32)
    plan.get_field(E)
    torch.cuda.synchronize()
    launches = plan.launch_count() - n0
    plan.destroy()
    return fd.cpu().numpy(), en.cpu().numpy(), E.cpu().numpy(), launches


@pytest.mark.parametrize("kind,order", [(LAG, 17), (LAG, 3), (LAG, 9), (LAG, 1), (SPL, 3)])
@pytest.mark.parametrize("Nx,Nv", [(64, 64), (256, 256), (128, 64), (64, 256), (256, 128)])
def test_small_run_against_the_oracle_steps(torch, vog, oracle, Nx, Nv, kind, order):
    """Unmerged XVX, 3 steps with an external field, delta-f (config 1's physics): state, field and energies against
    oracle.step; one launch for the whole run."""
    cfg = inputs.config(1, Nx=Nx, Nv=Nv, kind=kind, order=order)
    f0 = inputs.initial_f(cfg)
    n = 3
    rng = np.random.default_rng(7)
    ext = (0.02 * rng.standard_normal((n, cfg.Nx))).astype(np.float32)
    f, en, E, launches = _run(torch, vog, cfg, f0, n, ext, False, True)
    assert launches == 1
    fo = f0.astype(np.float64)
    feq = oracle.Feq.make(cfg.feq)
    eo = []
    for s in range(n):
        fo, Eo = oracle.step(fo, cfg.L, cfg.vmin, cfg.vmax, cfg.dt, cfg.kind, cfg.order, feq, cfg.split,
                             E_ext=ext[s].astype(np.float64))
        eo.append(oracle.electric_energy(Eo, cfg.L))
    assert np.abs(f - fo).max() <= 3 * n * TOL * _scale(f0, cfg)
    assert np.abs(E - Eo).max() <= 1e-5 * np.abs(Eo).max()
    assert np.abs(en - np.array(eo)).max() <= 1e-4 * max(eo)


@pytest.mark.parametrize("merge", [False, True])
@pytest.mark.parametrize("split", [0, 1])
@pytest.mark.parametrize("idx,over", [(0, {}), (1, {}), (2, {"Nx": 128, "Nv": 256}), (3, {"Nx": 256, "Nv": 64})])
def test_small_run_follows_the_kernel_per_launch_loop(torch, vog, idx, over, split, merge):
    """All four sequences (XVX / VXV, merged or not) on the four configs' physics (full f, delta-f, two Gaussians,
    driven from delta f = 0): the one-kernel run against the existing loop, 4 steps, E_ext, energies, final field."""
    cfg = inputs.config(idx, split=split, **over)
    f0 = inputs.initial_f(cfg)
    n = 4
    rng = np.random.default_rng(11)
    ext = (0.03 * rng.standard_normal((2 * n + 1, cfg.Nx))).astype(np.float32)
    f1, en1, E1, l1 = _run(torch, vog, cfg, f0, n, ext, merge, True)
    f2, en2, E2, l2 = _run(torch, vog, cfg, f0, n, ext, merge, False)
    assert l1 == 1 and l2 > 4 * n
    assert np.isfinite(f1).all()
    nadv = (2 * n + 1) if merge else 3 * n
    assert np.abs(f1.astype(np.float64) - f2).max() <= 2 * nadv * TOL * _scale(f0, cfg)
    escale = max(np.abs(E2).max(), np.abs(ext).max())
    assert np.abs(E1.astype(np.float64) - E2).max() <= 2e-5 * escale
    assert np.abs(en1 - en2).max() <= 2e-4 * max(en2.max(), 1e-30)


def test_small_run_vxv_reuses_the_field_of_the_previous_run(torch, vog):
    """VXV: the first half step of a run uses the field the previous run on the same array left in the plan."""
    cfg = inputs.config(1, split=1)
    f0 = inputs.initial_f(cfg)
    outs = []
    for small in (True, False):
        plan = vog.Plan.from_config(cfg)
        if small:
            plan.tune(29, 1)
        fd = _dev(torch, f0)
        plan.run(fd, cfg.dt, 2)
        plan.run(fd, cfg.dt, 3)
        torch.cuda.synchronize()
        outs.append(fd.cpu().numpy().astype(np.float64))
        plan.destroy()
    assert np.abs(outs[0] - outs[1]).max() <= 2 * 15 * TOL * np.abs(f0).max()


def test_small_run_repeats_bit_for_bit_and_rejects_large_grids(torch, vog):
    cfg = inputs.config(1)
    f0 = inputs.initial_f(cfg)
    a = _run(torch, vog, cfg, f0, 5, None, False, True)
    b = _run(torch, vog, cfg, f0, 5, None, False, True)
    assert np.array_equal(a[0], b[0]) and np.array_equal(a[1], b[1]) and np.array_equal(a[2], b[2])
    plan = vog.Plan(512, 64, 1.0, -1.0, 1.0)
    with pytest.raises(vog.VogError):
        plan.tune(29, 1)
    plan.destroy()
