"""vog_field_noalloc (include/vog.h): the field solve for callers that cannot allocate (scratch in a fixed device
array).  Its output against the existing plan-based path (vog_field), within the 2e-6 of max|E| that the field tests in
test_gpu_parity.py use, on two calls in a row.  In a file of its own that pytest collects last (the suite runs with
pytest -x).  Works alone in a fresh process and after the other tests: nothing here depends on earlier state, and the
second call uses a smaller grid than the first, so anything stale in the shared scratch would show.
"""
import numpy as np
import pytest

from paper_1301_5892_b200 import inputs

pytestmark = pytest.mark.gpu

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


def _existing_path(torch, vog, cfg, fd):
    plan = vog.Plan.from_config(cfg)
    E = torch.empty(cfg.Nx, device="cuda", dtype=torch.float32)
    plan.field(fd, E)
    torch.cuda.synchronize()
    out = E.cpu().numpy().astype(np.float64)
    plan.destroy()
    return out


def test_no_alloc_field_matches_the_plan_path_twice_in_a_row(torch, vog):
    cases = [inputs.config(2),                       # 1024 x 1024 bump on tail, delta-f
             inputs.config(1),                       # 256 x 256 nonlinear Landau, delta-f: smaller than the call before
             inputs.config(0, Nx=4096, Nv=64)]       # the maximum Nx, the minimum Nv, full f
    inputs_dev, outs, refs = [], [], []
    for cfg in cases:
        fd = torch.from_numpy(inputs.initial_f(cfg)).cuda()
        inputs_dev.append(fd)
        refs.append(_existing_path(torch, vog, cfg, fd))
    # the new entry point: calls back to back on one stream, no synchronisation between them, outputs pre-allocated
    Es = [torch.full((cfg.Nx,), float("nan"), device="cuda", dtype=torch.float32) for cfg in cases]
    for cfg, fd, E in zip(cases, inputs_dev, Es):
        vog.field_noalloc(fd, cfg.Nx, cfg.Nv, cfg.L, cfg.vmin, cfg.vmax, E)
    torch.cuda.synchronize()
    for cfg, E, ref in zip(cases, Es, refs):
        out = E.cpu().numpy().astype(np.float64)
        assert np.isfinite(out).all()
        scale = np.abs(ref).max()
        assert scale > 0
        # both paths are within 2e-6 of the oracle's field (test_gpu_parity.py): within 2 x 2e-6 of one another
        assert np.abs(out - ref).max() <= 2 * TOL * scale, (cfg.name, np.abs(out - ref).max() / scale)
        assert abs(out.mean()) <= TOL * scale            # zero mean
    # the same call again gives the same bits (the scratch carries nothing over)
    E2 = torch.empty_like(Es[0])
    vog.field_noalloc(inputs_dev[0], cases[0].Nx, cases[0].Nv, cases[0].L, cases[0].vmin, cases[0].vmax, E2)
    torch.cuda.synchronize()
    assert np.array_equal(E2.cpu().numpy(), Es[0].cpu().numpy())


def test_no_alloc_field_against_the_oracle(torch, vog, oracle):
    cfg = inputs.config(1)
    f = inputs.initial_f(cfg)
    E = torch.empty(cfg.Nx, device="cuda", dtype=torch.float32)
    vog.field_noalloc(torch.from_numpy(f).cuda(), cfg.Nx, cfg.Nv, cfg.L, cfg.vmin, cfg.vmax, E)
    torch.cuda.synchronize()
    Eo = oracle.field(f, cfg.L, cfg.vmin, cfg.vmax)
    assert np.abs(E.cpu().numpy() - Eo).max() <= TOL * np.abs(Eo).max()


def test_no_alloc_field_rejects_what_does_not_fit(torch, vog):
    f = torch.zeros((64, 8192), device="cuda", dtype=torch.float32)
    E = torch.zeros(8192, device="cuda", dtype=torch.float32)
    L = vog.lib()
    p = vog._ptr
    assert L.vog_field_noalloc(p(f), 8192, 64, 1.0, -1.0, 1.0, p(E), None) == vog.ETOOLARGE      # beyond the scratch
    assert "VOG_NOALLOC_MAX_NX" in vog.strerror(vog.ETOOLARGE)
    with pytest.raises(vog.VogError):
        vog.field_noalloc(f, 8192, 64, 1.0, -1.0, 1.0, E)
    assert L.vog_field_noalloc(p(f), 96, 64, 1.0, -1.0, 1.0, p(E), None) == vog.EINVAL            # not a power of two
    assert L.vog_field_noalloc(p(f), 64, 32, 1.0, -1.0, 1.0, p(E), None) == vog.EINVAL            # Nv too small
    assert L.vog_field_noalloc(None, 64, 64, 1.0, -1.0, 1.0, p(E), None) == vog.EINVAL
    assert L.vog_field_noalloc(p(f), 64, 64, 0.0, -1.0, 1.0, p(E), None) == vog.EINVAL
    assert L.vog_field_noalloc(p(f), 64, 64, 1.0, 1.0, 1.0, p(E), None) == vog.EINVAL
    assert vog.NOALLOC_MAX_NX == 4096
