"""Pins for the oracle (oracle/vog_oracle.c) against what the paper and the mathematics fix.

None of these retype the oracle's own formula: each compares the oracle with an
independent statement -- a closed form derived separately (Everett-form symbol), a library
routine (numpy.fft, numpy.interp, scipy CubicSpline / BarycentricInterpolator), an
invariant, a brute-force dense matrix, or the constant the paper prints.
SURVEY.md 8(c) pins P1-P7.
"""
import math
import os

import numpy as np
import pytest
from scipy.interpolate import BarycentricInterpolator, CubicSpline
from scipy.special import binom

from paper_1301_5892_b200 import inputs

LAG, SPL = 0, 1
KINDS = [(LAG, 1), (LAG, 3), (LAG, 5), (LAG, 9), (LAG, 17), (SPL, 3)]
GOLDEN = os.path.join(os.path.dirname(__file__), "golden")


def _golden(name):
    out = {}
    with open(os.path.join(GOLDEN, name)) as fh:
        for line in fh:
            if line.startswith("#") or not line.strip():
                continue
            key, val = line.split()
            out[key] = float(val)
    return out


# ---------------------------------------------------------------- P1: integer shifts
@pytest.mark.parametrize("kind,order", KINDS)
@pytest.mark.parametrize("b", [0, 1, -1, 5, -7, 64, -130, 1000003])
def test_integer_shift_is_exact_permutation(oracle, kind, order, b):
    """b* = 0 => u'_i = u_{(i+b) mod N}.  Lagrange: bit-exact."""
    rng = np.random.default_rng(1)
    N = 64
    u = rng.random(N)
    out = oracle.advect_line(u, float(b), kind, order)
    expect = u[(np.arange(N) + b) % N]
    if kind == LAG:
        assert np.array_equal(out, expect)
    else:  # spline goes through a linear solve: exact up to rounding only
        assert np.abs(out - expect).max() < 1e-14


def test_direction_positive_velocity_moves_profile_to_plus_x(oracle):
    """u(t,x) = u(s, x - c(t-s)): c > 0 => the bump moves toward +x."""
    N, L = 128, 2.0
    x = np.arange(N) * L / N
    u = np.exp(-200 * (x - 0.5) ** 2)
    f = np.tile(u, (4, 1))
    c = 3.0
    dt = 5 * (L / N) / c            # exactly five cells
    out = oracle.advect_x(f, L, c, c + 1e-9, dt, LAG, 17)   # v_0 = vmin = c
    assert np.argmax(out[0]) == np.argmax(u) + 5


def test_floor_split_for_negative_beta(oracle):
    assert oracle.split_shift(-0.25) == (-1, 0.75)
    assert oracle.split_shift(2.5) == (2, 0.5)
    assert oracle.split_shift(-3.0) == (-3, 0.0)


# ---------------------------------------------------------------- P2: Fourier mode, closed-form symbol
def _everett_P(s, t, d):
    """P(s;t) = sum_k C(t+k, 2k+1) (-s)^k, generalised binomial."""
    return sum(binom(t + k, 2 * k + 1) * (-s) ** k for k in range(d + 1))


def _symbol(kind, order, theta, beta):
    b = math.floor(beta)
    t = beta - b
    if kind == LAG:
        d = (order - 1) // 2
        s = 2 - 2 * math.cos(theta)
        return np.exp(1j * theta * b) * (_everett_P(s, 1 - t, d) + np.exp(1j * theta) * _everett_P(s, t, d))
    # cubic spline: cardinal B-spline values at t+1, t, t-1, t-2 over the collocation symbol (2+cos)/3
    Bm1 = (1 - t) ** 3 / 6
    B0 = (4 - 6 * t ** 2 + 3 * t ** 3) / 6
    B1 = (1 + 3 * t + 3 * t ** 2 - 3 * t ** 3) / 6
    B2 = t ** 3 / 6
    num = Bm1 * np.exp(-1j * theta) + B0 + B1 * np.exp(1j * theta) + B2 * np.exp(2j * theta)
    return np.exp(1j * theta * b) * num * 3 / (2 + math.cos(theta))


@pytest.mark.parametrize("kind,order", KINDS)
@pytest.mark.parametrize("beta", [0.37, -2.6, 7.999, 13.5, -0.001])
def test_fourier_mode_is_multiplied_by_closed_form_symbol(oracle, kind, order, beta):
    N = 96
    j = np.arange(N)
    for m in (0, 1, 5, 17, N // 2 - 1, N // 2):
        theta = 2 * math.pi * m / N
        phi = 0.3
        u = np.cos(theta * j + phi)
        lam = _symbol(kind, order, theta, beta)
        expect = abs(lam) * np.cos(theta * j + phi + np.angle(lam))
        out = oracle.advect_line(u, beta, kind, order)
        assert np.abs(out - expect).max() < 2e-13, (m, np.abs(out - expect).max())


# ---------------------------------------------------------------- P3: eigen-decomposition, N <= 16
@pytest.mark.parametrize("N", [8, 12, 16])
@pytest.mark.parametrize("beta", [0.25, -1.75, 3.5])
def test_dense_matrix_equals_circulant_eigendecomposition(oracle, N, beta):
    """A = U D U^*, U_{m,k} = e^{-2 i pi mk/N}, D = diag(FFT(a)); with the 1/N that
    makes U U^* = N I explicit (reading Q9)."""
    for d in (0, 1, 2):
        a = oracle.lagrange_first_row(N, d, beta)
        A = oracle.circulant(a)
        mk = np.outer(np.arange(N), np.arange(N))
        U = np.exp(-2j * np.pi * mk / N)
        D = np.diag(np.fft.fft(a))
        assert np.abs(U @ D @ U.conj().T / N - A).max() < 1e-14
        # and the paper's 4-step algorithm: FFT(D * FFT^{-1}(u))
        u = np.random.default_rng(N).random(N)
        assert np.abs(np.fft.fft(np.fft.fft(a) * np.fft.ifft(u)).real - A @ u).max() < 1e-14
        # stencil path == dense path
        assert np.abs(oracle.advect_line(u, beta, LAG, 2 * d + 1) - A @ u).max() < 1e-14


def test_circulant_layout_matches_eq4(oracle):
    """First row a_0 a_1 ..., second row a_{N-1} a_0 a_1 ...."""
    a = np.arange(5.0)
    A = oracle.circulant(a)
    assert np.array_equal(A[0], [0, 1, 2, 3, 4])
    assert np.array_equal(A[1], [4, 0, 1, 2, 3])
    assert np.array_equal(A[4], [1, 2, 3, 4, 0])


@pytest.mark.parametrize("beta", [0.0, 0.6, -2.3, 9.25])
def test_spline_dense_matrix_equals_line_solver(oracle, beta):
    """A = M x C(0..0,B(x_1),B(x_2),B(x_3))^{-1} by dense solves == cyclic-Thomas path."""
    N = 24
    A = oracle.spline_dense_matrix(N, 3, beta)
    u = np.random.default_rng(3).random(N)
    assert np.abs(A @ u - oracle.advect_line(u, beta, SPL, 3)).max() < 1e-13
    cc, _ = oracle.spline_first_rows(N, 3, beta)
    assert np.allclose(cc[-3:], [1 / 6, 4 / 6, 1 / 6]) and np.all(cc[:-3] == 0)


def test_even_degree_spline_collocation_is_singular_or_ill_conditioned(oracle):
    """Why "k=4" at P:227 is read as degree 3 / order 4 (reading Q6)."""
    N = 16
    cc, _ = oracle.spline_first_rows(N, 4, 0.3)
    assert np.linalg.cond(oracle.circulant(cc)) > 1e12
    cc3, _ = oracle.spline_first_rows(N, 3, 0.3)
    assert np.linalg.cond(oracle.circulant(cc3)) < 3.01


# ---------------------------------------------------------------- P4: library special cases
def test_bspline_recurrence_values(oracle):
    """Cox-de Boor against the textbook cubic pieces and partition of unity."""
    for t in (0.0, 0.2, 0.77):
        vals = [oracle.bspline(0, 3, j + t) for j in range(4)]
        expect = [t ** 3 / 6, (1 + 3 * t + 3 * t ** 2 - 3 * t ** 3) / 6,
                  (4 - 6 * t ** 2 + 3 * t ** 3) / 6, (1 - t) ** 3 / 6]
        assert np.allclose(vals, expect, atol=1e-15)
        assert abs(sum(vals) - 1) < 1e-15
    assert oracle.bspline(0, 3, 4.0) == 0.0 and oracle.bspline(0, 3, -0.1) == 0.0


def test_lag1_is_linear_interpolation(oracle):
    N = 50
    rng = np.random.default_rng(5)
    u = rng.random(N)
    for beta in (0.3, -4.2, 17.9):
        xq = (np.arange(N) + beta) % N
        ext = np.concatenate([u, u[:1]])
        expect = np.interp(xq, np.arange(N + 1), ext)
        assert np.abs(oracle.advect_line(u, beta, LAG, 1) - expect).max() < 1e-14


@pytest.mark.parametrize("order", [3, 9, 17])
def test_lagrange_matches_barycentric_interpolation_and_reproduces_polynomials(oracle, order):
    d = (order - 1) // 2
    for t in (0.0, 0.31, 0.5, 0.999):
        w = oracle.lagrange_weights(d, t)
        nodes = np.arange(-d, d + 2, dtype=float)
        assert abs(w.sum() - 1) < 1e-13
        # weights are the Lagrange basis at b*: compare with scipy on unit vectors
        for j in range(2 * d + 2):
            e = np.zeros(2 * d + 2)
            e[j] = 1
            assert abs(BarycentricInterpolator(nodes, e)(t) - w[j]) < 1e-11
        # degree <= p polynomials are reproduced exactly on a non-wrapping window
        for p in (0, 1, order):
            y = (nodes / (d + 1)) ** p
            assert abs(w @ y - (t / (d + 1)) ** p) < 1e-12


@pytest.mark.parametrize("beta", [0.4, -3.7, 11.25])
def test_cubic_spline_matches_scipy_periodic_spline(oracle, beta):
    N = 40
    rng = np.random.default_rng(7)
    u = rng.random(N)
    cs = CubicSpline(np.arange(N + 1), np.concatenate([u, u[:1]]), bc_type="periodic")
    expect = cs((np.arange(N) + beta) % N)
    assert np.abs(oracle.advect_line(u, beta, SPL, 3) - expect).max() < 1e-13


# ---------------------------------------------------------------- P5: invariants
@pytest.mark.parametrize("kind,order", KINDS)
def test_mass_is_conserved_to_1e12(oracle, kind, order):
    cfg = inputs.config(0, Nx=32, Nv=32, kind=kind, order=order)
    f = inputs.initial_f(cfg).astype(np.float64)
    m0 = f.sum()
    for _ in range(5):
        f, _E = oracle.step(f, cfg.L, cfg.vmin, cfg.vmax, cfg.dt, kind, order)
    assert abs(f.sum() - m0) / m0 < 1e-12


@pytest.mark.parametrize("kind,order", KINDS)
def test_v_advection_leaves_rho_unchanged_and_norm_does_not_grow(oracle, kind, order):
    rng = np.random.default_rng(11)
    Nx, Nv = 24, 48
    f = rng.random((Nv, Nx))
    E = rng.normal(size=Nx)
    g = oracle.advect_v(f, E, -6.0, 6.0, 0.7, kind, order)
    assert np.abs(oracle.density(g, -6, 6) - oracle.density(f, -6, 6)).max() < 1e-12
    # |lambda_m| <= 1 for odd-degree Lagrange and the cubic spline => l2 norm cannot grow
    assert np.linalg.norm(g) <= np.linalg.norm(f) * (1 + 1e-14)
    h = oracle.advect_x(f, 4 * math.pi, -6.0, 6.0, 0.7, kind, order)
    assert np.linalg.norm(h) <= np.linalg.norm(f) * (1 + 1e-14)
    assert abs(h.sum() - f.sum()) < 1e-10


def test_symbol_modulus_at_most_one():
    for kind, order in KINDS:
        for t in np.linspace(0, 0.999, 41):
            lam = [abs(_symbol(kind, order, 2 * math.pi * m / 256, t)) for m in range(129)]
            assert max(lam) <= 1 + 1e-12


def test_field_zero_mean_and_cosine_density(oracle):
    """mean(E) = 0; rho = cos(kx) => E = sin(kx)/k exactly (eq (2))."""
    Nx, L = 64, 4 * math.pi
    x = np.arange(Nx) * L / Nx
    for m in (1, 3, 9):
        k = 2 * math.pi * m / L
        E = oracle.poisson(1.0 + 0.2 * np.cos(k * x), L)
        assert abs(E.mean()) < 1e-15
        assert np.abs(E - 0.2 * np.sin(k * x) / k).max() < 1e-13
    # Nyquist content is dropped (reading Q12), a constant background too
    assert np.abs(oracle.poisson(5.0 + np.cos(math.pi * np.arange(Nx)), L)).max() < 1e-13


def test_field_equals_fft_solve(oracle):
    rng = np.random.default_rng(13)
    Nx, Nv, L = 128, 32, 7.0
    f = rng.random((Nv, Nx))
    rho = f.sum(axis=0) * (12.0 / Nv)
    rh = np.fft.fft(rho - rho.mean())
    k = 2 * np.pi * np.fft.fftfreq(Nx, d=L / Nx)
    Eh = np.zeros(Nx, complex)
    nz = (k != 0)
    Eh[nz] = rh[nz] / (1j * k[nz])
    Eh[Nx // 2] = 0
    expect = np.fft.ifft(Eh).real
    assert np.abs(oracle.field(f, L, -6.0, 6.0) - expect).max() < 1e-13
    assert abs(oracle.electric_energy(expect, L) - 0.5 * (L / Nx) * (expect ** 2).sum()) < 1e-15


def test_field_is_the_circular_convolution_with_its_green_function(oracle):
    """the Fourier solve is linear and translation invariant, so E = G (*) rho with G = the field of a unit point
    density; G is real, odd about cell 0 (1/(ik) is odd and imaginary), has zero mean, and its closed form is
    G_n = L/(pi Nx) sum_{m=1}^{Nx/2-1} sin(2 pi m n / Nx)/m (modes 0 and Nx/2 dropped, reading Q12).  The GPU path's
    x-space field solve (csrc: field_then_v) computes exactly this convolution; here the ORACLE is held to it."""
    rng = np.random.default_rng(21)
    Nx, L = 96, 5.0
    delta = np.zeros(Nx)
    delta[0] = 1.0
    G = oracle.poisson(delta, L)
    n = np.arange(Nx)
    closed = np.array([sum(math.sin(2 * math.pi * m * k / Nx) / m for m in range(1, Nx // 2)) for k in n]) * L / (math.pi * Nx)
    assert np.abs(G - closed).max() < 1e-13
    assert abs(G[0]) < 1e-15 and np.abs(G[1:] + G[:0:-1]).max() < 1e-14 and abs(G.mean()) < 1e-15
    rho = rng.random(Nx)
    conv = np.array([sum(G[(i - j) % Nx] * rho[j] for j in range(Nx)) for i in range(Nx)])
    assert np.abs(oracle.poisson(rho, L) - conv).max() < 1e-13
    # translation: shifting rho by 7 cells shifts E by 7 cells
    assert np.abs(oracle.poisson(np.roll(rho, 7), L) - np.roll(oracle.poisson(rho, L), 7)).max() < 1e-13


def test_delta_f_source_is_plain_difference(oracle):
    """P:197 with zero delta-f: the update is f_eq(v - dt E) - f_eq(v)."""
    cfg = inputs.config(1, Nx=16, Nv=32)
    feq = oracle.Feq.make(cfg.feq)
    E = np.linspace(-0.5, 0.5, 16)
    g = oracle.advect_v(np.zeros((32, 16)), E, cfg.vmin, cfg.vmax, 0.3, LAG, 17, feq)
    v = cfg.v()[:, None]
    expect = np.exp(-(v - 0.3 * E[None, :]) ** 2 / 2) / math.sqrt(2 * math.pi) - np.exp(-v ** 2 / 2) / math.sqrt(2 * math.pi)
    assert np.abs(g - expect).max() < 1e-15


# ---------------------------------------------------------------- P6 / P7: physics
def _landau_history(oracle, cfg, steps, use_feq, exact_f0=False):
    f = inputs.initial_f(cfg).astype(np.float64)
    if exact_f0:   # unrounded double initial condition (fp32 rounding of f0 alone moves the energy ~1e-5)
        f = (1.0 + cfg.alpha * np.cos(cfg.k * cfg.x()[None, :])) * inputs.gaussians(cfg.v()[:, None], cfg.profile)
        if cfg.feq:
            f = f - inputs.gaussians(cfg.v()[:, None], cfg.feq)
    feq = oracle.Feq.make(cfg.feq) if use_feq else None
    hist = []
    for _ in range(steps):
        f, _E = oracle.step(f, cfg.L, cfg.vmin, cfg.vmax, cfg.dt, cfg.kind, cfg.order, feq, cfg.split)
        hist.append(oracle.electric_energy(oracle.field(f, cfg.L, cfg.vmin, cfg.vmax), cfg.L))
    return np.array(hist)


def test_linear_landau_damping_rate(oracle):
    """Config 0: the field amplitude decays at gamma = 0.1533 (golden/landau_rate.txt)."""
    gamma = _golden("landau_rate.txt")["gamma"]
    cfg = inputs.config(0)
    ee = _landau_history(oracle, cfg, 100, False)
    t = cfg.dt * np.arange(1, 101)
    pk = [i for i in range(1, 99) if ee[i] > ee[i - 1] and ee[i] > ee[i + 1]]
    assert len(pk) >= 4
    slope = np.polyfit(t[pk], np.log(ee[pk]), 1)[0]
    assert abs(0.5 * slope + gamma) < 0.004, slope
    # oscillation frequency of the k=0.5 Langmuir wave, omega = 1.4156: energy peaks every pi/omega
    assert abs(np.mean(np.diff(t[pk])) - math.pi / 1.4156) < 0.05


def test_delta_f_scheme_matches_full_f_scheme_in_double(oracle):
    """different discretisations of the same v-step, equal to ~1e-8 of max energy."""
    cfg_full = inputs.config(0)
    cfg_df = inputs.config(0, feq=[(1 / math.sqrt(2 * math.pi), 0.0, 0.5)])
    a = _landau_history(oracle, cfg_full, 60, False, exact_f0=True)
    b = _landau_history(oracle, cfg_df, 60, True, exact_f0=True)
    assert np.abs(a - b).max() / a.max() < 1e-7


def test_split_orders_agree_on_landau_slope(oracle):
    cfg = inputs.config(0, split=inputs.SPLIT_VXV)
    f = inputs.initial_f(cfg).astype(np.float64)
    E = oracle.field(f, cfg.L, cfg.vmin, cfg.vmax)
    ee = []
    for _ in range(100):
        f, E = oracle.step(f, cfg.L, cfg.vmin, cfg.vmax, cfg.dt, cfg.kind, cfg.order, None, 1, None, E)
        ee.append(oracle.electric_energy(E, cfg.L))
    ee = np.array(ee)
    t = cfg.dt * np.arange(1, 101)
    pk = [i for i in range(1, 99) if ee[i] > ee[i - 1] and ee[i] > ee[i + 1]]
    slope = np.polyfit(t[pk], np.log(ee[pk]), 1)[0]
    assert abs(0.5 * slope + 0.1533) < 0.004


def test_keen_drive_matches_paper_parameters():
    g = _golden("keen_drive.txt")
    assert abs(inputs.keen_amplitude(g["t0"])) < 1e-15
    assert abs(inputs.keen_amplitude(g["tL"]) - 0.5) < 1e-3
    assert abs(inputs.keen_amplitude(200.0) - 1.0) < 1e-4
    cfg = inputs.config(3, Nx=64, Nv=64)
    e = inputs.keen_E_ext(cfg, 150.0)
    assert abs(np.abs(e).max() - g["Emax"] * g["k"] * inputs.keen_amplitude(150.0)) < 1e-3


# ---------------------------------------------------------------- round 2: E_ext in the step, f_eq with mu != 0
# (VERDICT r1 "What's weak" 2: flipping the sign of E_ext in oracle_step, or (v - mu) -> (v + mu) in oracle_feq,
# left every pin above green.  The pins below fix both by statements that are independent of the oracle's code:
# characteristics of the v-transport equation, translation of a profile, a Gaussian integral.)
_BUMP_FEQ = [(0.9 / math.sqrt(2 * math.pi), 0.0, 0.5), (0.2 / math.sqrt(2 * math.pi), 4.5, 4.0)]   # config 2's f_eq


@pytest.mark.parametrize("split", [inputs.SPLIT_XVX, inputs.SPLIT_VXV])
@pytest.mark.parametrize("kcells", [3, -5])
def test_step_with_constant_E_ext_is_a_pure_velocity_translation(oracle, split, kcells):
    """the advecting field is E + E_ext (E_ext = -E_app).  For f independent of x the self-consistent field
    vanishes and the x half steps act on constant lines, so one Strang step with a constant E_ext = c is the
    characteristic map f(v) -> f(v - c dt) (d_t f + E d_v f = 0).  With c dt = k dv (XVX; VXV: every half
    step k/2 cells... chosen even) this is the exact permutation f_new[j] = f[j - k]: c > 0 moves the profile to +v."""
    Nx, Nv, L, vmin, vmax, dt = 32, 64, 4 * math.pi, -6.0, 6.0, 0.1
    dv = (vmax - vmin) / Nv
    k = 2 * kcells                                   # even: the two VXV half steps are whole cells each
    c = k * dv / dt
    rng = np.random.default_rng(21)
    prof = rng.random(Nv)
    f = np.tile(prof[:, None], (1, Nx))
    E_ext = np.full(Nx, c)
    g, E = oracle.step(f, L, vmin, vmax, dt, LAG, 17, None, split, E_ext, np.zeros(Nx))
    assert np.abs(E).max() < 1e-13                   # rho is constant in x: zero-mean field vanishes
    expect = np.tile(np.roll(prof, k)[:, None], (1, Nx))     # f_new[j] = f[j - k]
    assert np.abs(g - expect).max() < 1e-13
    # and the opposite sign must NOT satisfy it (guards the test itself against a symmetric profile)
    assert np.abs(g - np.tile(np.roll(prof, -k)[:, None], (1, Nx))).max() > 0.1


def test_step_xvx_with_E_ext_cancelling_the_self_field_is_two_x_half_steps(oracle):
    """P:269 again: with E_ext = -E_self the advecting field is zero, the v-advection is the identity (beta = 0
    is an exact permutation) and the XVX step is x(dt/2) twice."""
    cfg = inputs.config(0, Nx=32, Nv=32)
    f = inputs.initial_f(cfg).astype(np.float64)
    half = oracle.advect_x(f, cfg.L, cfg.vmin, cfg.vmax, 0.5 * cfg.dt, LAG, 17)
    E_self = oracle.field(half, cfg.L, cfg.vmin, cfg.vmax)
    assert np.abs(E_self).max() > 1e-5
    g, E = oracle.step(f, cfg.L, cfg.vmin, cfg.vmax, cfg.dt, LAG, 17, None, inputs.SPLIT_XVX, -E_self)
    expect = oracle.advect_x(half, cfg.L, cfg.vmin, cfg.vmax, 0.5 * cfg.dt, LAG, 17)
    assert np.array_equal(E, E_self)
    assert np.abs(g - expect).max() < 1e-15
    # with +E_self instead the field doubles and the result must differ
    g2, _ = oracle.step(f, cfg.L, cfg.vmin, cfg.vmax, cfg.dt, LAG, 17, None, inputs.SPLIT_XVX, E_self)
    assert np.abs(g2 - expect).max() > 1e-7


@pytest.mark.parametrize("split", [inputs.SPLIT_XVX, inputs.SPLIT_VXV])
def test_step_delta_f_source_sees_E_ext_with_its_sign(oracle, split):
    """delta-f mode with delta f = 0 and a constant E_ext = c: the step returns f_eq(v - c dt) - f_eq(v), the
    TRANSLATED equilibrium profile (two-Gaussian f_eq of config 2, mu = 4.5): sampled on an unwrapped extension of
    the v mesh and shifted by whole cells -- no formula of the oracle is re-evaluated."""
    Nx, Nv, L, vmin, vmax, dt, k = 32, 256, 20 * math.pi, -9.0, 9.0, 0.05, 6
    dv = (vmax - vmin) / Nv
    c = k * dv / dt
    ext = vmin + dv * np.arange(-16, Nv + 16)                      # unwrapped mesh, 16 cells beyond either end
    prof = inputs.gaussians(ext, _BUMP_FEQ)
    expect = prof[16 - k:16 - k + Nv] - prof[16:16 + Nv]           # f_eq(v_j - k dv) - f_eq(v_j)
    g, _E = oracle.step(np.zeros((Nv, Nx)), L, vmin, vmax, dt, LAG, 17, oracle.Feq.make(_BUMP_FEQ), split,
                        np.full(Nx, c), np.zeros(Nx))
    # VXV takes two half steps: source(k/2) shifted by k/2 cells + source(k/2) = the same total, up to the Lagrange
    # interpolation error of the intermediate (smooth, dv-resolved) profile, ~1e-9 here (LAG17, Nv = 256)
    tol = 1e-15 if split == inputs.SPLIT_XVX else 1e-12
    assert np.abs(g - expect[:, None]).max() < tol
    assert np.abs(g + expect[:, None]).max() > 1e-3                # the mirrored sign fails


def test_feq_two_gaussians_off_centre(oracle):
    """oracle_feq with n = 2, mu != 0 (config 2, B.json): position of the bump, mirror symmetry of each Gaussian
    about ITS centre, the Gaussian integral sum_g amp_g sqrt(pi / c_g) (closed form; the rectangle rule is
    spectrally accurate for a Gaussian), and agreement with the profile the workload generator builds f_0 from."""
    feq = oracle.Feq.make(_BUMP_FEQ)
    v = -9.0 + (18.0 / 1024) * np.arange(1024)
    val = np.array([oracle.feq_eval(feq, x) for x in v])
    assert oracle.feq_eval(feq, 4.5) > 50 * oracle.feq_eval(feq, -4.5)        # the bump sits at +4.5, not -4.5
    bump_only = oracle.Feq.make(_BUMP_FEQ[1:])
    for h in (0.1, 0.37, 1.0):
        assert abs(oracle.feq_eval(bump_only, 4.5 + h) - oracle.feq_eval(bump_only, 4.5 - h)) < 1e-17
        assert oracle.feq_eval(bump_only, 4.5) > oracle.feq_eval(bump_only, 4.5 + h)
    closed = sum(a * math.sqrt(math.pi / c) for a, _mu, c in _BUMP_FEQ)        # = 0.9 + 0.2 / sqrt(8)
    assert abs(closed - (0.9 + 0.2 / math.sqrt(8.0))) < 1e-15
    assert abs(val.sum() * (18.0 / 1024) - closed) < 1e-12
    first_moment = sum(a * mu * math.sqrt(math.pi / c) for a, mu, c in _BUMP_FEQ)
    assert abs((val * v).sum() * (18.0 / 1024) - first_moment) < 1e-12        # odd in the sign of mu
    assert np.abs(val - inputs.gaussians(v, _BUMP_FEQ)).max() < 1e-16


def test_delta_f_source_with_off_centre_feq_is_a_translated_profile(oracle):
    """P:197 for config 2's f_eq: delta f = 0, E dt = k dv  =>  the update is f_eq sampled k cells lower minus f_eq."""
    Nx, Nv, vmin, vmax, dt = 4, 512, -9.0, 9.0, 0.05
    dv = (vmax - vmin) / Nv
    ks = np.array([7, -3, 0, 12])
    E = ks * dv / dt
    ext = vmin + dv * np.arange(-16, Nv + 16)
    prof = inputs.gaussians(ext, _BUMP_FEQ)
    g = oracle.advect_v(np.zeros((Nv, Nx)), E, vmin, vmax, dt, LAG, 17, oracle.Feq.make(_BUMP_FEQ))
    for i, k in enumerate(ks):
        expect = prof[16 - k:16 - k + Nv] - prof[16:16 + Nv]
        assert np.abs(g[:, i] - expect).max() < 2e-16


def test_delta_f_scheme_matches_full_f_scheme_with_off_centre_feq(oracle):
    """P:197-199 on a bump-on-tail shaped state: advancing delta f = f - f_eq and adding f_eq back equals advancing f,
    up to the interpolation error of f_eq itself (LAG17 on a dv-resolved Gaussian: ~1e-9)."""
    cfg = inputs.config(2, Nx=32, Nv=512)
    v = cfg.v()[:, None]
    f_full = (1.0 + cfg.alpha * np.cos(cfg.k * cfg.x()[None, :])) * inputs.gaussians(v, cfg.profile)
    feq_v = inputs.gaussians(v, cfg.feq)
    E = 0.6 * np.sin(cfg.k * cfg.x()) + 0.3                                   # |E dt / dv| up to ~1.3 cells
    a = oracle.advect_v(f_full, E, cfg.vmin, cfg.vmax, cfg.dt, LAG, 17, None)
    b = oracle.advect_v(f_full - feq_v, E, cfg.vmin, cfg.vmax, cfg.dt, LAG, 17, oracle.Feq.make(cfg.feq))
    assert np.abs(a - (b + feq_v)).max() < 1e-8
    # sanity of the bound: the source term itself is 4 orders larger than the tolerance
    assert np.abs(b - oracle.advect_v(f_full - feq_v, E, cfg.vmin, cfg.vmax, cfg.dt, LAG, 17, None)).max() > 1e-4


def test_keen_drive_sign_and_phase(oracle):
    """the advecting field is E - E_app with E_app = E_max k a(t) sin(kx - w t); the harness passes
    E_ext = -E_app.  Pins the SIGN and the phase velocity (+w/k) of inputs.keen_E_ext, not only its modulus."""
    g = _golden("keen_drive.txt")
    cfg = inputs.config(3, Nx=256, Nv=64)
    x = cfg.x()
    for t in (100.0, 150.0, 200.0):
        e = inputs.keen_E_ext(cfg, t).astype(np.float64)
        a = inputs.keen_amplitude(t)
        assert a > 0
        # projection on sin(kx - wt): -E_max k a(t) (negative: E_ext = -E_app), nothing on the cosine
        s, c = np.sin(g["k"] * x - g["omega"] * t), np.cos(g["k"] * x - g["omega"] * t)
        assert abs(2 * (e * s).mean() + g["Emax"] * g["k"] * a) < 1e-8
        assert abs(2 * (e * c).mean()) < 1e-8
    # the pattern travels toward +x at w/k: the zero crossing with negative slope of E_ext... follows x = w t / k
    t0, t1 = 150.0, 150.5
    ph = lambda t: np.angle(np.fft.fft(inputs.keen_E_ext(cfg, t).astype(np.float64))[1])
    dphi = (ph(t1) - ph(t0) + math.pi) % (2 * math.pi) - math.pi
    assert abs(dphi + g["omega"] * (t1 - t0)) < 1e-6          # mode e^{i(kx - wt)}: phase of FFT bin 1 falls at w
    # driven particles: with f independent of x and NO self field, a step with E_ext(t) moves the column at the
    # maximum of E_ext toward +v (characteristics dv/dt = E + E_ext)
    i = int(np.argmax(e))
    Nv = 64
    prof = np.exp(-np.linspace(-3, 3, Nv) ** 2)
    f = np.tile(prof[:, None], (1, 256))
    dt = 4 * cfg.dv / float(e[i])                               # four cells at the maximum
    out, _ = oracle.step(f, cfg.L, cfg.vmin, cfg.vmax, dt, LAG, 17, None, inputs.SPLIT_VXV, e, np.zeros(256))
    assert np.argmax(out[:, i]) == np.argmax(prof) + 4


# ---------------------------------------------------------------- NEXT-3: trapezoid field solve and diagnostics
def test_trapezoid_field_on_a_mode_has_the_closed_form_factor(oracle):
    """rho = 1 + a cos(kx): summing the trapezoid rule in closed form gives E = a sin(kx)/k * (k dx/2)/tan(k dx/2),
    i.e. the Fourier solve's answer times 1 - (k dx)^2/12 + O((k dx)^4), and the zero-mean
    modifications leave exactly that."""
    L = 4 * math.pi
    for Nx, m in ((32, 1), (64, 3), (256, 5)):
        dx = L / Nx
        x = np.arange(Nx) * dx
        k = 2 * math.pi * m / L
        E = oracle.field_trapezoid(1.0 + 0.3 * np.cos(k * x), L)
        fac = (k * dx / 2) / math.tan(k * dx / 2)
        assert np.abs(E - 0.3 * fac * np.sin(k * x) / k).max() < 1e-13
        assert abs(E.mean()) < 1e-15
        assert abs(fac - (1 - (k * dx) ** 2 / 12)) < (k * dx) ** 4 / 100
        Ef = oracle.poisson(1.0 + 0.3 * np.cos(k * x), L)
        assert abs(np.abs(E).max() / np.abs(Ef).max() - fac) < 1e-12


def test_trapezoid_field_without_zero_mean_keeps_the_systematic_error(oracle):
    """without the modification rho~ = rho - 1; a density whose mean is 1 + eps (the rounding drift the
    paper talks about) then leaves a ramp eps x in E, which the zero-mean version removes."""
    Nx, L, eps = 128, 4 * math.pi, 1e-4
    x = np.arange(Nx) * L / Nx
    rho = 1.0 + eps + 0.01 * np.cos(0.5 * x)
    E0 = oracle.field_trapezoid(rho, L, zero_mean=False, background=1.0)
    E1 = oracle.field_trapezoid(rho, L, zero_mean=True)
    ramp = E0 - oracle.field_trapezoid(rho - eps, L, zero_mean=False, background=1.0)
    assert np.abs(ramp - eps * x).max() < 1e-13
    assert abs(E1.mean()) < 1e-16
    assert np.abs(E1 - oracle.field_trapezoid(rho - eps, L, zero_mean=True)).max() < 1e-13   # the mean plays no role
    # Poisson's equation holds cell by cell for the trapezoid rule: (E_{k+1} - E_k)/dx = mean of rho~ over the cell
    d = np.diff(E1) / (L / Nx)
    rt = rho - rho.mean()
    assert np.abs(d - 0.5 * (rt[:-1] + rt[1:])).max() < 1e-13


def test_rho_modes_and_kinetic_energy_closed_forms(oracle):
    """rho^_0 and |rho^_1| against numpy.fft; the kinetic energy of a Maxwellian is L/2 (second moment 1),
    the rectangle rule being spectrally accurate for a Gaussian."""
    rng = np.random.default_rng(3)
    rho = 1.0 + 0.1 * rng.normal(size=96)
    r0, r1 = oracle.rho_modes(rho)
    F = np.fft.fft(rho) / rho.size
    assert abs(r0 - F[0].real) < 1e-15 and abs(r1 - abs(F[1])) < 1e-15
    assert abs(oracle.rho_modes(1.0 + 0.25 * np.cos(2 * math.pi * np.arange(64) / 64 + 0.7))[1] - 0.125) < 1e-15
    cfg = inputs.config(0, Nx=32, Nv=256, vmin=-8.0, vmax=8.0)
    f = np.tile((np.exp(-cfg.v() ** 2 / 2) / math.sqrt(2 * math.pi))[:, None], (1, 32))
    assert abs(oracle.kinetic_energy(f, cfg.L, cfg.vmin, cfg.vmax) - 0.5 * cfg.L) < 1e-12
    # weights: doubling one row's value adds (1/2) dx dv v_j^2 * (row sum)
    g = f.copy()
    g[40] *= 2
    dx, dv = cfg.L / 32, 16.0 / 256
    assert abs(oracle.kinetic_energy(g, cfg.L, -8, 8) - oracle.kinetic_energy(f, cfg.L, -8, 8)
               - 0.5 * dx * dv * cfg.v()[40] ** 2 * f[40].sum()) < 1e-15
