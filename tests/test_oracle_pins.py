"""Pins of the CPU oracle against what the paper and the mathematics fix.

None of these retype the oracle's formulas: each compares the oracle with a closed form, an invariant,
a dense-matrix brute force built here with numpy, or a library routine (numpy.fft, scipy.linalg.expm).
"""
import os

import numpy as np
import pytest
import scipy.linalg

from paper_1204_5434_b200 import inputs

GOLD = os.path.join(os.path.dirname(__file__), "golden")


# ------------------------------------------------------------------ FFT ----------
@pytest.mark.parametrize("n", [1, 2, 4, 6, 8, 15, 16, 32, 64])
def test_fft_matches_definition_and_numpy(oracle, n):
    rng = np.random.default_rng(n)
    x = rng.normal(size=n) + 1j * rng.normal(size=n)
    X = oracle.fft1d(x, -1)
    assert np.max(np.abs(X - oracle.dft1d_direct(x, -1))) < 1e-13 * n
    assert np.max(np.abs(X - np.fft.fft(x))) < 1e-13 * n                       # sign convention e^{-ikx}
    assert np.max(np.abs(oracle.fft1d(X, +1) - x)) < 1e-13                     # F^-1 F = I, 1/n on the inverse
    assert abs(np.sum(np.abs(X) ** 2) / n - np.sum(np.abs(x) ** 2)) < 1e-12 * n   # Parseval


# ------------------------------------------------------------------ uniform field ---------------
@pytest.mark.parametrize("w0", [0.7, 0.3 - 1.1j])
def test_uniform_field_closed_form(oracle, w0):
    """q_j = exp(-w0 j ds), Q = exp(-w0), phi = 1 (north_star; closed form of PAPER.md Eq. 4-5)."""
    grid, Ns = (4, 8, 2), 16
    o = oracle.Oracle(grid, (3.0, 4.0, 5.0), Ns, "external")
    o.set_fields(np.full(grid, w0, np.complex128))
    o.propagate()
    Q, phi, _ = o.density_operators()
    assert abs(Q - np.exp(-w0)) < 1e-14
    assert np.max(np.abs(phi - 1.0)) < 1e-13
    for j in (0, 1, 7, Ns):
        assert np.max(np.abs(o.get_slice(0, j) - np.exp(-w0 * j / Ns))) < 1e-14


def test_uniform_diblock_closed_form(oracle):
    grid, Ns, fA = (4, 4, 4), 20, 0.3
    wp, wm = 0.4 + 0.2j, -0.6 + 0.1j
    o = oracle.Oracle(grid, (4.0, 4.0, 4.0), Ns, "diblock", fA=fA, chiN=15.0)
    o.set_fields(np.full(grid, wp, np.complex128), np.full(grid, wm, np.complex128))
    o.propagate()
    Q, pa, pb = o.density_operators()
    wA, wB = wp - wm, wp + wm
    assert abs(Q - np.exp(-(fA * wA + (1 - fA) * wB))) < 1e-14
    assert np.max(np.abs(pa - fA)) < 1e-13 and np.max(np.abs(pb - (1 - fA))) < 1e-13


# ------------------------------------------------------------------ dense brute force -----------
def _dense_dft(n):
    k = np.arange(n)
    return np.exp(-2j * np.pi * np.outer(k, k) / n)


def _dense_k2(grid, cell):
    ks = []
    for n, L in zip(grid, cell):
        i = np.arange(n)
        ks.append(2 * np.pi * np.where(i <= n // 2, i, i - n) / L)
    KX, KY, KZ = np.meshgrid(*ks, indexing="ij")
    return (KX ** 2 + KY ** 2 + KZ ** 2).ravel()


def _dense_F(grid):
    return np.kron(np.kron(_dense_dft(grid[0]), _dense_dft(grid[1])), _dense_dft(grid[2]))


@pytest.mark.parametrize("grid,cell", [((4, 4, 4), (3.0, 4.0, 5.0)), ((2, 8, 4), (2.0, 6.0, 3.5))])
def test_rqm4_step_equals_dense_operator(oracle, grid, cell):
    """Eq. 12 multiplied out as dense M x M matrices."""
    M = int(np.prod(grid))
    ds = 0.05
    w = inputs.random_complex_field(grid, 1, scale=0.8, mean=0.3).ravel()
    q = (1.0 + inputs.random_complex_field(grid, 2, scale=0.5)).ravel()
    F = _dense_F(grid)
    Fi = np.conj(F).T / M
    k2 = _dense_k2(grid, cell)
    D = lambda a: Fi @ np.diag(np.exp(-a * k2 * ds)) @ F
    E = lambda a: np.diag(np.exp(-a * w * ds))
    full = E(0.5) @ D(1.0) @ E(0.5)
    half = E(0.25) @ D(0.5) @ E(0.5) @ D(0.5) @ E(0.25)
    U = (4.0 * half - full) / 3.0
    got = oracle.rqm4_step(grid, cell, ds, w.reshape(grid), q.reshape(grid)).ravel()
    assert np.max(np.abs(got - U @ q)) < 1e-13


def test_converges_to_matrix_exponential_order4(oracle):
    """q(s=1) -> expm(Laplacian_spectral - diag w) 1 on 4^3, error falling ~16x per doubling of Ns."""
    grid, cell = (4, 4, 4), (3.0, 4.0, 5.0)
    M = 64
    w = inputs.random_complex_field(grid, 3, scale=1.0, mean=0.5)
    F = _dense_F(grid)
    lap = (np.conj(F).T / M) @ np.diag(-_dense_k2(grid, cell)) @ F
    exact = scipy.linalg.expm(lap - np.diag(w.ravel())) @ np.ones(M)
    errs = []
    for Ns in (16, 32, 64, 128, 256):
        o = oracle.Oracle(grid, cell, Ns, "external")
        o.set_fields(w)
        o.propagate()
        errs.append(np.max(np.abs(o.get_slice(0, Ns).ravel() - exact)))
    ratios = [errs[i] / errs[i + 1] for i in range(4)]
    assert errs[-1] < 1e-8
    assert all(12.0 < r < 17.0 for r in ratios), (errs, ratios)     # rough field: 12.7, 14.1, 15, 15.5 -> 16
    assert ratios[-1] > 15.0


def test_order4_at_config1(oracle):
    """Q(Ns) - Q(512) falls 16x per halving of ds on the config-1 field (PAPER.md:122 'globally fourth-order')."""
    cfg = inputs.config1()
    Qs = {}
    for Ns in (8, 16, 32, 64, 512):
        o = oracle.Oracle(cfg.grid, cfg.cell, Ns, "external")
        o.set_fields(cfg.f0)
        o.propagate()
        Qs[Ns] = o.density_operators()[0]
    errs = [abs(Qs[n] - Qs[512]) for n in (8, 16, 32, 64)]
    ratios = [errs[i] / errs[i + 1] for i in range(3)]
    assert all(12.0 < r < 18.0 for r in ratios), (errs, ratios)


# ------------------------------------------------------------------ invariants ------------------
@pytest.mark.parametrize("model", ["external", "diblock"])
def test_qqdag_invariant_and_normalisation(oracle, model):
    """(1/M) sum_x q_j q+_{Ns-j} = Q for every j (bilinear product, reading A-9); mean phi_A = fA, mean phi = 1."""
    if model == "diblock":
        cfg = inputs.small_diblock(grid=(4, 8, 16), Ns=20, fA=0.4)
        o = oracle.Oracle(cfg.grid, cfg.cell, cfg.Ns, "diblock", fA=cfg.fA, chiN=cfg.chiN)
        o.set_fields(cfg.f0, cfg.f1)
    else:
        cfg = inputs.config1(grid=(8, 8, 8), Ns=16)
        o = oracle.Oracle(cfg.grid, cfg.cell, cfg.Ns, "external")
        o.set_fields(cfg.f0)
    o.propagate()
    Q, pa, pb = o.density_operators()
    for j in range(cfg.Ns + 1):
        Qj = np.mean(o.get_slice(0, j) * o.get_slice(1, cfg.Ns - j))
        assert abs(Qj - Q) < 1e-13 * abs(Q), j
    assert abs(np.mean(o.get_slice(1, cfg.Ns)) - Q) < 1e-13 * abs(Q)            # Q[q+] = Q[q]
    if model == "diblock":
        assert abs(np.mean(pa) - cfg.fA) < 1e-12 and abs(np.mean(pa + pb) - 1.0) < 1e-12
    else:
        assert abs(np.mean(pa) - 1.0) < 1e-12


# ------------------------------------------------------------------ Debye response --------------
def _gD(x):
    return 2.0 * (np.exp(-x) + x - 1.0) / x ** 2


@pytest.mark.parametrize("n", [(1, 0, 0), (0, 1, 1), (2, 1, 0)])
def test_debye_response_homopolymer(oracle, n):
    """phi - 1 = -eps g_D(k^2) cos(k.x) for w = eps cos(k.x)   (north_star g_D)."""
    grid, cell, Ns, eps = (16, 16, 16), (4.0, 4.0, 4.0), 64, 1e-4
    X = np.meshgrid(*[np.arange(g) * (L / g) for g, L in zip(grid, cell)], indexing="ij")
    th = 2 * np.pi * sum(n[d] * X[d] / cell[d] for d in range(3))
    o = oracle.Oracle(grid, cell, Ns, "external")
    o.set_fields((eps * np.cos(th)).astype(np.complex128))
    o.propagate()
    _, phi, _ = o.density_operators()
    coef = 2.0 * np.mean((phi.real - 1.0) * np.cos(th))
    k2 = sum((2 * np.pi * n[d] / cell[d]) ** 2 for d in range(3))
    assert abs(coef / (-eps * _gD(k2)) - 1.0) < 2e-6


def test_debye_response_diblock_blocks(oracle):
    """Block-resolved response: phi_A - fA = -eps (g_AA + g_AB) cos, phi_A + phi_B - 1 = -eps g_D cos
    for wA = wB = eps cos (textbook diblock Debye functions; pins the jA split and per-block Simpson)."""
    grid, cell, Ns, fA, eps = (16, 1, 1), (4.0, 1.0, 1.0), 60, 0.3, 1e-4
    x = np.arange(16) * (4.0 / 16)
    th = (2 * np.pi * x / 4.0).reshape(grid)
    o = oracle.Oracle(grid, cell, Ns, "diblock", fA=fA, chiN=10.0)
    o.set_fields((eps * np.cos(th)).astype(np.complex128), np.zeros(grid, np.complex128))
    o.propagate()
    _, pa, pb = o.density_operators()
    k2 = (2 * np.pi / 4.0) ** 2
    gAA = 2.0 * (np.exp(-fA * k2) + fA * k2 - 1.0) / k2 ** 2
    gAB = (1 - np.exp(-fA * k2)) * (1 - np.exp(-(1 - fA) * k2)) / k2 ** 2
    cA = 2.0 * np.mean((pa.real - fA) * np.cos(th))
    cT = 2.0 * np.mean((pa.real + pb.real - 1.0) * np.cos(th))
    assert abs(cA / (-eps * (gAA + gAB)) - 1.0) < 2e-6
    assert abs(cT / (-eps * _gD(k2)) - 1.0) < 2e-6
    assert abs(oracle.debye(k2) - _gD(k2)) < 1e-15 and abs(oracle.debye(0.0) - 1.0) < 1e-15
    from decimal import Decimal, getcontext
    getcontext().prec = 60
    for xs in ("0.00005", "0.009", "0.011", "0.5"):                                  # both branches vs 60-digit arithmetic
        xd = Decimal(xs)
        ref = 2 * ((-xd).exp() + xd - 1) / (xd * xd)
        assert abs(oracle.debye(float(xs)) - float(ref)) < 1e-11


# ------------------------------------------------------------------ saddles and field updates ---
def test_diblock_homogeneous_saddle(oracle):
    """W- = chiN(2fA-1)/2, any uniform W+: both forces vanish, H/CV = -chiN(1-2fA)^2/4."""
    grid, Ns, fA, chiN = (4, 4, 4), 20, 0.3, 16.0
    wm, wp = chiN * (2 * fA - 1) / 2, 0.37
    o = oracle.Oracle(grid, (4.0,) * 3, Ns, "diblock", fA=fA, chiN=chiN)
    o.set_fields(np.full(grid, wp, np.complex128), np.full(grid, wm, np.complex128))
    H, resid = o.scft_step(5.0, 5.0, seidel=1)
    assert abs(H - (-chiN * (1 - 2 * fA) ** 2 / 4)) < 1e-13
    assert resid[0] < 1e-13 and resid[1] < 1e-13
    a, b = o.get_fields()
    assert np.max(np.abs(a - wp)) < 1e-12 and np.max(np.abs(b - wm)) < 1e-12


@pytest.mark.parametrize("seidel", [0, 1])
def test_scft_relaxes_to_mean_field_solution(oracle, seidel):
    """1-D lamellar: residuals of the mean-field equations fall and H drops below the homogeneous value."""
    grid, cell, Ns, fA, chiN = (32, 1, 1), (4.0, 1.0, 1.0), 40, 0.5, 20.0
    x = np.arange(32) * (4.0 / 32)
    wm = (2.0 * np.cos(2 * np.pi * x / 4.0)).reshape(grid).astype(np.complex128)
    o = oracle.Oracle(grid, cell, Ns, "diblock", fA=fA, chiN=chiN)
    o.set_fields(np.zeros(grid, np.complex128), wm)
    res = []
    for _ in range(80):
        H, r = o.scft_step(5.0, 5.0, seidel=seidel)
        res.append(max(r))
    assert res[-1] < 1e-3 and res[-1] < 1e-2 * res[0]
    assert H.real < -chiN * (1 - 2 * fA) ** 2 / 4 - 0.1 and abs(H.imag) < 1e-12
    a, b = o.get_fields()
    assert np.max(np.abs(a.imag)) < 1e-12 and np.max(np.abs(b.imag)) < 1e-12      # Wick-rotated fields stay real


@pytest.mark.parametrize("scheme", [0, 1])
def test_edwards_noise_free_relaxation_reaches_saddle(oracle, scheme):
    """Omega* = -iC/B, Q = exp(-C/B), mu = ln C + C/B, Pi = C + C^2/(2B)   (Eq. 2 as printed, reading A-13/A-14)."""
    grid, Ns, B, Cc = (8, 8, 8), 8, 2.0, 3.0
    rng = np.random.default_rng(5)
    om = -1j * Cc / B + 0.05 * rng.normal(size=grid)
    o = oracle.Oracle(grid, (4.0,) * 3, Ns, "edwards", B=B, Cc=Cc, noise_scale=0.0)
    o.set_fields(om.astype(np.complex128))
    for it in range(200):
        o.cl_step(0.2, scheme, 1, it)
    f, _ = o.get_fields()
    assert np.max(np.abs(f - (-1j * Cc / B))) < 1e-9
    o.propagate()
    Q, _, _ = o.density_operators()
    H, mu, Pi = o.operators()
    assert abs(Q - np.exp(-Cc / B)) < 1e-9
    assert abs(mu - (np.log(Cc) + Cc / B)) < 1e-9
    assert abs(Pi - (Cc + Cc ** 2 / (2 * B))) < 1e-8


def _block_debye(fA, k2):
    """Textbook diblock Debye functions g_AA, g_BB, g_AB at x = k^2 Rg^2 (same forms as test_debye_response_diblock_blocks)."""
    fB = 1.0 - fA
    gAA = 2.0 * (np.exp(-fA * k2) + fA * k2 - 1.0) / k2 ** 2
    gBB = 2.0 * (np.exp(-fB * k2) + fB * k2 - 1.0) / k2 ** 2
    gAB = (1 - np.exp(-fA * k2)) * (1 - np.exp(-fB * k2)) / k2 ** 2
    return gAA, gBB, gAB


@pytest.mark.parametrize("n,dtp,dtm", [(1, 5.0, 5.0), (2, 0.7, 2.5), (3, 12.0, 0.3)])
def test_scft_step_is_the_semi_implicit_step_of_the_linearised_dynamics(oracle, n, dtp, dtm):
    """Pins the two multipliers of the SCFT update (reading A-10; Eq. 10-11 at zero noise).

    Around the homogeneous state (fA = 1/2, W- = 0) a single mode eps*cos(kx) has the linear-response forces
    F+ = -g_D(k^2) W+ and F- = (2/chiN - S(k^2)) W-, S = g_AA + g_BB - 2 g_AB.  Eq. 11 treats g_D (for
    W+) and 2/chiN (for W-) implicitly, so ONE step must give the backward-Euler / IMEX amplitudes
        W+' = W+ / (1 + dt+ g_D),      W-' = W- (1 + dt- S) / (1 + 2 dt-/chiN)
    up to O(eps^2) and the O(ds^4) contour error.  A denominator 1 + dt+ or 1 + dt-*2 fails this at every (k, dt)."""
    grid, cell, Ns, fA, chiN, eps = (16, 1, 1), (4.0, 1.0, 1.0), 64, 0.5, 12.0, 1e-5
    x = np.arange(16) * (4.0 / 16)
    c = np.cos(2 * np.pi * n * x / 4.0).reshape(grid)
    k2 = (2 * np.pi * n / 4.0) ** 2
    gAA, gBB, gAB = _block_debye(fA, k2)
    o = oracle.Oracle(grid, cell, Ns, "diblock", fA=fA, chiN=chiN)
    o.set_fields((eps * c).astype(np.complex128), np.zeros(grid, np.complex128))
    o.scft_step(dtp, dtm, seidel=0)
    a, b = o.get_fields()
    amp = 2.0 * np.mean(a.real * c)
    assert abs(amp / eps - 1.0 / (1.0 + dtp * _gD(k2))) < 2e-6
    assert np.max(np.abs(a - amp * c)) < 1e-3 * eps and np.max(np.abs(b)) < 1e-3 * eps      # no other mode, W- untouched
    o.set_fields(np.zeros(grid, np.complex128), (eps * c).astype(np.complex128))
    o.scft_step(dtp, dtm, seidel=0)
    a, b = o.get_fields()
    amp = 2.0 * np.mean(b.real * c)
    S = gAA + gBB - 2.0 * gAB
    assert abs(amp / eps - (1.0 + dtm * S) / (1.0 + 2.0 * dtm / chiN)) < 2e-6
    assert np.max(np.abs(b - amp * c)) < 1e-3 * eps and np.max(np.abs(a)) < 1e-3 * eps


def _k2_grid(grid, cell):
    ks = [2 * np.pi * np.fft.fftfreq(g, d=L / g) for g, L in zip(grid, cell)]
    KX, KY, KZ = np.meshgrid(*ks, indexing="ij")
    return KX ** 2 + KY ** 2 + KZ ** 2


def _gD_safe(x):
    x = np.asarray(x, float)
    out = np.ones_like(x)
    nz = x > 1e-8
    out[nz] = 2.0 * (np.exp(-x[nz]) + x[nz] - 1.0) / x[nz] ** 2
    return out


@pytest.mark.parametrize("n,dt", [(1, 0.3), (3, 1.7)])
def test_cl_scheme1_edwards_is_backward_euler_and_filters_the_noise(oracle, n, dt):
    """Pins cl_step scheme=1, Edwards branch (reading A-11; Eq. 10-11).

    (a) noise off, Omega = Omega* + eps cos(kx): the linearised force is (B + C g_D(k^2)) dOmega (chain feels i*Omega),
        Eq. 10 treats exactly that operator implicitly, so one step gives dOmega' = dOmega / (1 + l dt (B + C g_D)).
    (b) noise on, AT the saddle (force identically zero): solving Eq. 10 for the new field divides the noise by the same
        operator, dOmega^(k) = eta^(k) / (1 + l dt (B + C g_D(k^2))), with eta = sqrt(2 l dt/dV) N(0,1) (the normals and
        their amplitude are pinned separately above).  Undivided noise (Eq. 11 as printed) fails (b)."""
    grid, cell, Ns, B, Cc, lam, eps = (16, 1, 1), (4.0, 1.0, 1.0), 64, 2.0, 3.0, 0.8, 1e-5
    x = np.arange(16) * (4.0 / 16)
    c = np.cos(2 * np.pi * n * x / 4.0).reshape(grid)
    k2 = (2 * np.pi * n / 4.0) ** 2
    o = oracle.Oracle(grid, cell, Ns, "edwards", B=B, Cc=Cc, lambda_plus=lam, noise_scale=0.0)
    o.set_fields((-1j * Cc / B + eps * c).astype(np.complex128))
    o.cl_step(dt, 1, 1, 0)
    f, _ = o.get_fields()
    amp = 2.0 * np.mean((f - (-1j * Cc / B)).real * c)
    assert abs(amp / eps - 1.0 / (1.0 + lam * dt * (B + Cc * _gD(k2)))) < 2e-6
    grid3, cell3 = (4, 8, 2), (3.0, 4.0, 5.0)
    M = int(np.prod(grid3))
    o = oracle.Oracle(grid3, cell3, 8, "edwards", B=B, Cc=Cc, lambda_plus=lam)
    o.set_fields(np.full(grid3, -1j * Cc / B, np.complex128))
    o.cl_step(dt, 1, 11, 5)
    f, _ = o.get_fields()
    eta = np.sqrt(2 * lam * dt / (np.prod(cell3) / M)) * np.array([oracle.normal(11, 5, 0, i) for i in range(M)]).reshape(grid3)
    want = np.fft.ifftn(np.fft.fftn(eta) / (1.0 + lam * dt * (B + Cc * _gD_safe(_k2_grid(grid3, cell3)))))
    assert np.max(np.abs((f - (-1j * Cc / B)) - want)) < 1e-12
    assert np.max(np.abs((f - (-1j * Cc / B)) - eta)) > 1e-3                         # the filter is not a no-op here


def test_cl_scheme1_diblock_is_backward_euler_and_filters_the_noise(oracle):
    """Pins cl_step scheme=1, diblock branch (reading A-11): W+ implicit in C g_D(k^2), W- implicit in 2C/chiN.

    (a) noise off, W+ = eps cos(kx) on the fA = 1/2 homogeneous state: F+ = -g_D W+, so W+' = W+/(1 + l+ dt C g_D);
        W- = eps cos: W-' = W- (1 + l- dt C S)/(1 + 2 l- dt C/chiN), S = g_AA + g_BB - 2 g_AB.
    (b) noise on at the homogeneous saddle W- = chiN(2fA-1)/2 (both forces vanish, test_diblock_homogeneous_saddle):
        dW+ = i F^-1{eta+^/(1 + l+ dt C g_D)},  dW- = eta-/(1 + 2 l- dt C/chiN)."""
    grid, cell, Ns, fA, chiN, Cc, lp, lm, dt, eps = (16, 1, 1), (4.0, 1.0, 1.0), 64, 0.5, 12.0, 4.0, 0.7, 1.3, 0.4, 1e-5
    x = np.arange(16) * (4.0 / 16)
    c = np.cos(2 * np.pi * 2 * x / 4.0).reshape(grid)
    k2 = (2 * np.pi * 2 / 4.0) ** 2
    gAA, gBB, gAB = _block_debye(fA, k2)
    kw = dict(fA=fA, chiN=chiN, Cc=Cc, lambda_plus=lp, lambda_minus=lm)
    o = oracle.Oracle(grid, cell, Ns, "diblock", noise_scale=0.0, **kw)
    o.set_fields((eps * c).astype(np.complex128), np.zeros(grid, np.complex128))
    o.cl_step(dt, 1, 1, 0)
    a, _ = o.get_fields()
    assert abs(2.0 * np.mean(a.real * c) / eps - 1.0 / (1.0 + lp * dt * Cc * _gD(k2))) < 2e-6
    o.set_fields(np.zeros(grid, np.complex128), (eps * c).astype(np.complex128))
    o.cl_step(dt, 1, 1, 0)
    _, b = o.get_fields()
    S = gAA + gBB - 2.0 * gAB
    assert abs(2.0 * np.mean(b.real * c) / eps - (1.0 + lm * dt * Cc * S) / (1.0 + 2.0 * lm * dt * Cc / chiN)) < 2e-6
    grid3, cell3, fA3 = (4, 2, 8), (3.0, 4.0, 5.0), 0.3
    M = int(np.prod(grid3))
    wm, wp = chiN * (2 * fA3 - 1) / 2, 0.21
    o = oracle.Oracle(grid3, cell3, 20, "diblock", fA=fA3, chiN=chiN, Cc=Cc, lambda_plus=lp, lambda_minus=lm)
    o.set_fields(np.full(grid3, wp, np.complex128), np.full(grid3, wm, np.complex128))
    o.cl_step(dt, 1, 21, 9)
    a, b = o.get_fields()
    dV = np.prod(cell3) / M
    ep = np.sqrt(2 * lp * dt / dV) * np.array([oracle.normal(21, 9, 0, i) for i in range(M)]).reshape(grid3)
    em = np.sqrt(2 * lm * dt / dV) * np.array([oracle.normal(21, 9, 1, i) for i in range(M)]).reshape(grid3)
    want_p = 1j * np.fft.ifftn(np.fft.fftn(ep) / (1.0 + lp * dt * Cc * _gD_safe(_k2_grid(grid3, cell3))))
    assert np.max(np.abs((a - wp) - want_p)) < 1e-12
    assert np.max(np.abs((b - wm) - em / (1.0 + 2.0 * lm * dt * Cc / chiN))) < 1e-12


def test_edwards_H_at_the_homogeneous_saddle(oracle):
    """Eq. 2 as printed (reading A-13) at Omega* = -iC/B: (B/2) V Omega*^2 = -C^2 V/(2B), ln Q = -C/B,
    so H = -C^2 V/(2B) + C^2 V/B = C^2 V/(2B); mu = ln C + C/B."""
    grid, cell, B, Cc = (4, 8, 2), (3.0, 4.0, 5.0), 2.5, 3.0
    V = float(np.prod(cell))
    o = oracle.Oracle(grid, cell, 8, "edwards", B=B, Cc=Cc)
    o.set_fields(np.full(grid, -1j * Cc / B, np.complex128))
    o.propagate()
    H, mu, _ = o.operators()
    assert abs(H - Cc ** 2 * V / (2 * B)) < 1e-12 * V
    assert abs(mu - (np.log(Cc) + Cc / B)) < 1e-13


def test_pressure_kernel_matches_volume_derivative_of_lnQ(oracle):
    """-(2/3V) K = d ln Q / dV at fixed lattice fields (reading A-14), one species: q+ = q.  The diblock branch has its own pin below."""
    cfg = inputs.config1(grid=(8, 8, 8), Ns=64)
    V = float(np.prod(cfg.cell))

    def lnQ(scale):
        cell = tuple(L * scale ** (1 / 3) for L in cfg.cell)
        o = oracle.Oracle(cfg.grid, cell, cfg.Ns, "external")
        o.set_fields(cfg.f0)
        o.propagate()
        return np.log(o.density_operators()[0]), o

    d = 1e-4
    fd = (lnQ(1 + d)[0] - lnQ(1 - d)[0]) / (2 * d * V)
    _, o = lnQ(1.0)
    _, _, Pi = o.operators()                     # model 0: Pi = -(2/3) K
    assert abs(Pi / V - fd) < 5e-3 * abs(fd)


def test_diblock_pressure_matches_volume_derivative_of_lnQ(oracle):
    """The diblock branch Pi = C - (2C/3) K (reading A-14) with complex fields and unequal blocks, where q+ is NOT q: the
    K term must still be the volume derivative of ln Q at fixed lattice fields, (Pi - C)/(C V) = -(2/3V) K = d ln Q / dV.
    The pin tells q+_{Ns-j} from q_{Ns-j} (and from q+_j): K rebuilt from the oracle's own slices with either slip misses the
    finite difference by far more than the tolerance."""
    def case(Ns):
        cfg = inputs.small_diblock(grid=(8, 8, 8), cell=(3.0, 3.5, 4.0), Ns=Ns, fA=0.25, complex_fields=True)
        V, Cc = float(np.prod(cfg.cell)), cfg.C

        def solve(scale):
            cell = tuple(L * scale ** (1 / 3) for L in cfg.cell)
            o = oracle.Oracle(cfg.grid, cell, cfg.Ns, "diblock", fA=cfg.fA, chiN=cfg.chiN, B=cfg.B, Cc=Cc)
            o.set_fields(cfg.f0, cfg.f1)
            o.propagate()
            return np.log(o.density_operators()[0]), o

        d = 1e-4
        fd = (solve(1 + d)[0] - solve(1 - d)[0]) / (2 * d * V)
        _, o = solve(1.0)
        _, _, Pi = o.operators()
        return cfg, V, o, fd, (Pi - Cc) / (Cc * V)

    # K is the derivative of the contour-continuous ln Q; the lattice ln Q converges to it with the contour step
    # (measured: relative gap 4.0e-2, 5.9e-3, 6.6e-4, 5.7e-5 at Ns = 16, 32, 64, 128)
    _, _, _, fd32, got32 = case(32)
    cfg, V, o, fd, got = case(64)
    assert abs(fd.imag) > 1e-3 * abs(fd.real) > 0            # genuinely complex: a conjugation slip would show
    assert abs(got - fd) < 1e-3 * abs(fd), (got, fd)
    assert abs(got - fd) / abs(fd) < 0.2 * abs(got32 - fd32) / abs(fd32)
    # discriminating power: the same contour sum with q_{Ns-j} or q+_j in place of q+_{Ns-j}
    Ns, jA = cfg.Ns, int(round(cfg.fA * cfg.Ns))
    k = [2 * np.pi * np.fft.fftfreq(n, L / n) for n, L in zip(cfg.grid, cfg.cell)]
    k2 = k[0][:, None, None] ** 2 + k[1][None, :, None] ** 2 + k[2][None, None, :] ** 2
    simpson = lambda n: np.array([1.0] + [4.0 if i % 2 else 2.0 for i in range(1, n)] + [1.0]) / 3.0
    c = np.zeros(Ns + 1); c[:jA + 1] += simpson(jA); c[jA:] += simpson(Ns - jA)
    Q = o.density_operators()[0]

    def K_of(partner):
        tot = 0.0
        for j in range(Ns + 1):
            lap = np.fft.ifftn(-k2 * np.fft.fftn(o.get_slice(0, j)))
            tot += c[j] * np.mean(partner(j) * lap)
        return tot / (Ns * Q)

    right = -(2.0 / (3.0 * V)) * K_of(lambda j: o.get_slice(1, Ns - j))
    assert abs(right - fd) < 1e-3 * abs(fd)
    for slip in (lambda j: o.get_slice(0, Ns - j), lambda j: o.get_slice(1, j)):
        wrong = -(2.0 / (3.0 * V)) * K_of(slip)
        assert abs(wrong - fd) > 2e-2 * abs(fd)


# ------------------------------------------------------------------ Philox / noise --------------
def test_philox_known_answers(oracle):
    rows = [l.split() for l in open(os.path.join(GOLD, "philox4x32_10_kat.txt")) if l.strip() and not l.startswith("#")]
    assert len(rows) == 3
    for r in rows:
        v = [int(t, 16) for t in r]
        assert oracle.philox4x32_10(v[0:4], v[4:6]) == tuple(v[6:10])


def test_normal_moments_and_noise_amplitude(oracle):
    n = 200000
    z = np.array([oracle.normal(99, 3, 1, i) for i in range(n)])
    assert abs(z.mean()) < 4 / np.sqrt(n)
    assert abs(z.var() - 1.0) < 4 * np.sqrt(2.0 / n)
    assert abs(np.mean(z ** 4) - 3.0) < 4 * np.sqrt(96.0 / n)
    assert oracle.normal(99, 3, 1, 5) != oracle.normal(99, 3, 0, 5) != oracle.normal(99, 4, 0, 5)
    # Var eta = 2 lambda dt / dV: one Edwards CL step from a force-free state of B=0, C->0
    grid, cell, dt = (8, 8, 8), (2.0, 2.0, 2.0), 0.01
    o = oracle.Oracle(grid, cell, 4, "edwards", B=0.0, Cc=1e-300, lambda_plus=1.0)
    o.set_fields(np.zeros(grid, np.complex128))
    o.cl_step(dt, 0, 7, 0)
    f, _ = o.get_fields()
    dV = 8.0 / 512
    assert np.max(np.abs(f.imag)) < 1e-200
    assert abs(f.real.var() / (2 * dt / dV) - 1.0) < 4 * np.sqrt(2.0 / 512)
    assert f.real.ravel()[5] == pytest.approx(np.sqrt(2 * dt / dV) * oracle.normal(7, 0, 0, 5), rel=1e-15)


def test_cl_step_diblock_euler_maruyama_signs(oracle):
    """Zero-noise EM step equals W+ + dt C (phiA+phiB-1), W- - dt C (2W-/chiN + phiB - phiA)."""
    cfg = inputs.small_diblock(grid=(4, 4, 8), Ns=8, fA=0.5)
    kw = dict(fA=cfg.fA, chiN=cfg.chiN, Cc=cfg.C)
    o = oracle.Oracle(cfg.grid, cfg.cell, cfg.Ns, "diblock", noise_scale=0.0, **kw)
    o.set_fields(cfg.f0, cfg.f1)
    o.propagate()
    _, pa, pb = o.density_operators()
    o.cl_step(0.01, 0, 1, 0)
    a, b = o.get_fields()
    assert np.max(np.abs(a - (cfg.f0 + 0.01 * cfg.C * (pa + pb - 1)))) < 1e-14
    assert np.max(np.abs(b - (cfg.f1 - 0.01 * cfg.C * (2 * cfg.f1 / cfg.chiN + pb - pa)))) < 1e-14
    # with noise: W+ gets i*eta, W- gets eta, independent streams (reading A-15)
    o2 = oracle.Oracle(cfg.grid, cfg.cell, cfg.Ns, "diblock", **kw)
    o2.set_fields(cfg.f0, cfg.f1)
    o2.cl_step(0.01, 0, 42, 3)
    a2, b2 = o2.get_fields()
    M = int(np.prod(cfg.grid))
    amp = np.sqrt(2 * 0.01 / (np.prod(cfg.cell) / M))
    ep = np.array([oracle.normal(42, 3, 0, i) for i in range(M)]).reshape(cfg.grid)
    em = np.array([oracle.normal(42, 3, 1, i) for i in range(M)]).reshape(cfg.grid)
    assert np.max(np.abs((a2 - a) - 1j * amp * ep)) < 1e-13
    assert np.max(np.abs((b2 - b) - amp * em)) < 1e-13


def test_fp32_oracle_tracks_fp64(oracle):
    cfg = inputs.config1(grid=(8, 8, 8), Ns=16)
    Qs = []
    for prec in ("f64", "f32"):
        o = oracle.Oracle(cfg.grid, cfg.cell, cfg.Ns, "external", precision=prec)
        o.set_fields(cfg.f0)
        o.propagate()
        Qs.append(o.density_operators()[0])
    assert abs(Qs[1] - Qs[0]) < 2e-5 * abs(Qs[0])


def test_create_rejects_bad_arguments(oracle):
    with pytest.raises(ValueError):
        oracle.Oracle((4, 4, 4), (1.0,) * 3, 10, "diblock", fA=0.33)     # fA*Ns not an integer (reading A-4)
    with pytest.raises(ValueError):
        oracle.Oracle((4, 4, 4), (1.0,) * 3, 10, "diblock", fA=0.5)      # odd block (Simpson, reading A-5)
    with pytest.raises(ValueError):
        oracle.Oracle((4, 4, 4), (1.0,) * 3, 7, "external")


# ------------------------------------------------------------------------------------------------
# linear multiblock chains (oracle_set_blocks)
# ------------------------------------------------------------------------------------------------
def _solve_blocks(oracle, cfg, blocks=None, f0=None, f1=None, model="diblock"):
    kw = dict(fA=cfg.fA, chiN=cfg.chiN, B=cfg.B, Cc=cfg.C)
    o = oracle.Oracle(cfg.grid, cfg.cell, cfg.Ns, model, **kw)
    if blocks is not None:
        o.set_blocks(*blocks)
    o.set_fields(cfg.f0 if f0 is None else f0, cfg.f1 if f1 is None else f1)
    o.propagate()
    return o, o.density_operators()


def test_multiblock_pins(oracle):
    """What fixes the block machinery without another implementation: (i) chain reversal - listing the blocks from the other
    end swaps the roles of q and q+ and must leave Q, phi_A, phi_B unchanged (a wrong segment index for q+ breaks it);
    (ii) two A blocks of even length are one homopolymer: Q and phi_A equal the one-species model in w_A = W+ - W-, phi_B = 0
    (pins the junction weights 1/3 + 1/3 = 2/3 of Simpson per block, reading A-5); (iii) an ABA triblock obeys
    mean q_j q+_{Ns-j} = Q for every j, mean phi_A = its A fraction and phi_A + phi_B averages to 1; in a uniform field
    phi_A is identically that fraction; (iv) the two-block list reproduces the default diblock bit for bit."""
    from paper_1204_5434_b200 import inputs
    cfg = inputs.small_diblock(grid=(8, 4, 8), cell=(3.0, 4.0, 5.0), Ns=12, fA=0.5)
    _, (Q0, a0, b0) = _solve_blocks(oracle, cfg)
    _, (Q1, a1, b1) = _solve_blocks(oracle, cfg, ([0, 1], [6, 6]))
    assert Q0 == Q1 and np.array_equal(a0, a1) and np.array_equal(b0, b1)                                  # (iv)
    for blocks, rev in ((([0, 1], [4, 8]), ([1, 0], [8, 4])), (([0, 1, 0], [2, 6, 4]), ([0, 1, 0], [4, 6, 2])),
                        (([1, 0, 1, 0], [2, 2, 4, 4]), ([0, 1, 0, 1], [4, 4, 2, 2]))):
        _, (Qa, aa, ba) = _solve_blocks(oracle, cfg, blocks)
        _, (Qb, ab, bb) = _solve_blocks(oracle, cfg, rev)
        assert abs(Qa - Qb) < 1e-13 * abs(Qa) and np.max(np.abs(aa - ab)) < 1e-13 and np.max(np.abs(ba - bb)) < 1e-13      # (i)
    _, (Qh, ah, bh) = _solve_blocks(oracle, cfg, ([0, 0], [4, 8]))                                          # (ii)
    oe = oracle.Oracle(cfg.grid, cfg.cell, cfg.Ns, "external")
    oe.set_fields(cfg.f0 - cfg.f1); oe.propagate()
    Qe, ae, _ = oe.density_operators()
    assert abs(Qh - Qe) < 1e-14 * abs(Qe) and np.max(np.abs(ah - ae)) < 1e-13 and np.max(np.abs(bh)) == 0.0
    o, (Qt, at, bt) = _solve_blocks(oracle, cfg, ([0, 1, 0], [2, 6, 4]))                                    # (iii)
    for j in range(cfg.Ns + 1):
        assert abs(np.mean(o.get_slice(0, j) * o.get_slice(1, cfg.Ns - j)) - Qt) < 1e-13 * abs(Qt), j
    assert abs(np.mean(at) - 0.5) < 1e-13 and abs(np.mean(at + bt) - 1.0) < 1e-13
    w0 = 0.3 - 0.2j
    _, (Qu, au, bu) = _solve_blocks(oracle, cfg, ([0, 1, 0], [2, 6, 4]), f0=np.full(cfg.grid, w0), f1=np.zeros(cfg.grid, complex))
    assert abs(Qu - np.exp(-w0)) < 1e-14 and np.max(np.abs(au - 0.5)) < 1e-13 and np.max(np.abs(bu - 0.5)) < 1e-13
    with pytest.raises(RuntimeError):
        oracle.Oracle(cfg.grid, cfg.cell, cfg.Ns, "diblock", fA=0.5).set_blocks([0, 1], [5, 7])             # odd blocks: no Simpson
    with pytest.raises(RuntimeError):
        oracle.Oracle(cfg.grid, cfg.cell, cfg.Ns, "external").set_blocks([0], [12])
