"""GPU tests of the in-place v-advection (vog_shift_v / vog_advect_v with Nv >= 1024; csrc/vog_os2.cuh osv7_kernel in
its whole-strip mode, csrc/vog_os.cu strip_copy_kernel; vog_plan_tune(34, 0/1)).

A strip whose integer shifts are at most 24 rows is stored in place: the store of a pair of blocks waits until the
windows of its neighbours are on chip, the strip's first rows, which the last window reads again after the wrap, are
kept in shared memory, and the rows on either side of a piece of work that is not a whole strip are saved in a global
scratch before any CTA starts such a piece (shapes below: 4096 x 1024 has left-over strips cut into shares, 512 x 8192
four CTAs per strip).  Other strips go through the plan's second grid and are copied back.  The arithmetic per pair
of blocks is that of the out-of-place kernel, so the result must be BIT-IDENTICAL to vog_shift_v_to on the same input,
whatever the mix of strips (up to rounding in a column's last pair of blocks, see _same); against the oracle it is checked at the
usual 2e-6 of max|f| (BASELINE.json north_star).
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


def _dev(torch, a):
    return torch.from_numpy(np.ascontiguousarray(a)).cuda()


def _same(torch, g, out, Nv, ikind):
    """Bit-identical, except in the last pair of blocks of a column: its window runs past the last row and, behind the
    saved first rows, reads rows that may already have been advanced; those samples only reach discarded outputs, but
    they go through the same complex transform as the pair's kept samples, whose outputs then move by rounding (a few
    1e-7 of max|f|)."""
    V = 228 if ikind == 1 else 232
    nb = (Nv + V - 1) // V
    last = ((nb + 1) // 2 * 2 - 2) * V                  # first row of the last pair of blocks
    if not torch.equal(g[:last], out[:last]):
        return False
    return float((g[last:] - out[last:]).abs().max()) <= 1e-6 * float(out.abs().max())


def _betas(Nx, kind, seed):
    rng = np.random.default_rng(seed)
    if kind == "small":            # every strip in place
        return rng.uniform(-8.0, 8.0, Nx)
    if kind == "edge":             # around the limit of 24 rows: strips on either side of it
        return rng.uniform(-30.0, 30.0, Nx)
    if kind == "negative":         # large negative shifts stay in place (only the wrap after the last row is bounded)
        return rng.uniform(-90.0, 5.0, Nx)
    if kind == "lowedge":          # strips whose first window just fits / just misses the rows kept below a piece
        b = np.empty(Nx)
        for s0 in range(0, Nx, 16):
            lo = [-33.5, -31.5, -27.5, -25.5, -23.5, -19.5][(s0 // 16) % 6]
            b[s0:s0 + 16] = lo + rng.uniform(0.0, 6.0, 16)
        return b
    if kind == "mixed":            # some strips far outside (second grid), some with a wide spread (per-lane landing)
        b = rng.uniform(-6.0, 6.0, Nx)
        b[Nx // 8:Nx // 4] += 300.0
        b[Nx // 2:Nx // 2 + 16] = rng.uniform(-400.0, 400.0, 16)
        b[-16:] -= 1000.5
        return b
    raise ValueError(kind)


@pytest.mark.parametrize("kind", ["small", "edge", "lowedge", "negative", "mixed"])
@pytest.mark.parametrize("Nx,Nv,ikind,order", [(2048, 2048, 0, 17), (4096, 1024, 0, 9), (1024, 4096, 1, 3), (512, 8192, 0, 3)])
def test_inplace_v_is_bit_identical_to_out_of_place(torch, vog, Nx, Nv, ikind, order, kind):
    rng = np.random.default_rng(5)
    f = rng.random((Nv, Nx), dtype=np.float32)
    beta = _betas(Nx, kind, 11)
    plan = vog.Plan(Nx, Nv, 1.0, -1.0, 1.0, ikind, order)
    fd = _dev(torch, f)
    out = torch.empty_like(fd)
    bd = _dev(torch, beta)
    plan.shift_v_to(fd, out, bd)
    for rep in range(2):                        # twice: the second call sees whatever flags the first one left
        g = fd.clone()
        plan.shift_v(g, bd)
        torch.cuda.synchronize()
        assert _same(torch, g, out, Nv, ikind), "call %d" % rep
    # the copy-everything path gives the same bits
    plan.tune(34, 0)
    g = fd.clone()
    plan.shift_v(g, bd)
    torch.cuda.synchronize()
    assert torch.equal(g, out)
    plan.destroy()


@pytest.mark.parametrize("kind", ["small", "mixed"])
def test_inplace_v_against_the_oracle(torch, vog, oracle, kind):
    Nx, Nv = 256, 2048
    f = inputs.smooth_grid(Nx, Nv).astype(np.float32)
    beta = _betas(Nx, kind, 3)
    plan = vog.Plan(Nx, Nv, 1.0, -1.0, 1.0, 0, 17)
    fd = _dev(torch, f)
    plan.shift_v(fd, _dev(torch, beta))
    torch.cuda.synchronize()
    ref = oracle.shift_v(f.astype(np.float64), beta, 0, 17)
    assert np.abs(fd.cpu().numpy() - ref).max() <= TOL * np.abs(f).max()
    plan.destroy()


@pytest.mark.parametrize("shape", [None, (4096, 1024), (512, 4096)])
def test_inplace_advect_v_with_source_matches_the_step_kernel(torch, vog, oracle, shape):
    """vog_advect_v (delta-f source included) in place against the oracle's advect_v: the bench grid (whole strips), a
    grid with left-over strips cut into shares and one with several CTAs per strip."""
    cfg = inputs.metric_config() if shape is None else inputs.config(1, Nx=shape[0], Nv=shape[1])
    f = inputs.initial_f(cfg)
    rng = np.random.default_rng(2)
    E = (0.3 * np.sin(2 * np.pi * np.arange(cfg.Nx) / cfg.Nx) + 0.05 * rng.standard_normal(cfg.Nx)).astype(np.float32)
    plan = vog.Plan.from_config(cfg)
    fd = _dev(torch, f)
    plan.advect_v(fd, _dev(torch, E), cfg.dt)
    torch.cuda.synchronize()
    ref = oracle.advect_v(f.astype(np.float64), E.astype(np.float64), cfg.vmin, cfg.vmax, cfg.dt, cfg.kind, cfg.order,
                          oracle.Feq.make(cfg.feq))
    scale = max(float(np.abs(f).max()), 1e-2)
    assert np.abs(fd.cpu().numpy() - ref).max() <= TOL * scale
    plan.destroy()


@pytest.mark.timeout(300)
def test_inplace_v_on_several_streams_at_once(torch, vog):
    """In-place calls of three plans on three streams share the GPU: no CTA may wait for another CTA of its grid to
    become resident (an earlier version synchronised the halo saving through a counter inside the kernel and would hang
    here: each grid holds SMs the other grids' remaining CTAs need).  Results as for one stream."""
    Nx, Nv = 4096, 4096
    rng = np.random.default_rng(9)
    beta = _dev(torch, rng.uniform(-8.0, 8.0, Nx))
    streams = [torch.cuda.Stream() for _ in range(3)]
    plans = [vog.Plan(Nx, Nv, 1.0, -1.0, 1.0, 0, 17, stream=s) for s in streams]
    f0 = torch.rand((Nv, Nx), device="cuda")
    ref = torch.empty_like(f0)
    plans[0].shift_v_to(f0, ref, beta)
    torch.cuda.synchronize()
    fs = [f0.clone() for _ in plans]
    torch.cuda.synchronize()
    for p_, f_ in zip(plans, fs):
        p_.shift_v(f_, beta)
    torch.cuda.synchronize()
    for f_ in fs:
        assert _same(torch, f_, ref, Nv, 0)
    for rep in range(10):                        # and again, back to back on all three
        for p_, f_ in zip(plans, fs):
            p_.shift_v(f_, beta)
    torch.cuda.synchronize()
    for p_ in plans:
        p_.destroy()
