"""GPU parity: the CUDA path (through the C-ABI) against the CPU oracle, element by element, same seeded inputs.

Tolerances (BASELINE.json north_star): fp64 1e-11 relative on Q, 1e-9 max-abs on phi and q(r,1);
fp32 2e-4 relative; CL trajectories with identical Philox noise 1e-8 after 10 steps (fp64).
"""
import numpy as np
import pytest
import torch

from paper_1204_5434_b200 import inputs

pytestmark = pytest.mark.gpu


@pytest.fixture(scope="module")
def B():
    assert torch.cuda.is_available(), "these tests need a CUDA device"
    from paper_1204_5434_b200 import binding
    binding.lib()
    return binding


def _dev(a, dtype=torch.complex128):
    return torch.from_numpy(np.ascontiguousarray(a)).to("cuda:0").to(dtype).contiguous()


def _kw(cfg):
    return dict(fA=cfg.fA, chiN=cfg.chiN, B=cfg.B, Cc=cfg.C)


def _pair(B, oracle, cfg, precision="f64", store_both=1, **extra):
    """store_both = 1 (every slice kept) unless the test is about the default meet-in-the-middle store."""
    kw = _kw(cfg); kw.update(extra)
    dt = torch.complex128 if precision == "f64" else torch.complex64
    g = B.Fts(cfg.grid, cfg.cell, cfg.Ns, cfg.model, precision=precision, store_both=store_both, **kw)
    o = oracle.Oracle(cfg.grid, cfg.cell, cfg.Ns, cfg.model, precision="f64", **kw)    # the fp64 oracle judges both precisions
    f1 = None if cfg.f1 is None else _dev(cfg.f1, dt)
    g.set_fields(_dev(cfg.f0, dt), f1)
    o.set_fields(cfg.f0, cfg.f1)
    return g, o


def _cmp_solve(g, o, tolQ, tolphi, two):
    g.propagate(); o.propagate()
    Qg, pa, pb = g.density_operators()
    Qo, oa, ob = o.density_operators()
    assert abs(Qg - Qo) <= tolQ * abs(Qo), (Qg, Qo)
    assert np.max(np.abs(pa.cpu().numpy() - oa)) <= tolphi
    if two:
        assert np.max(np.abs(pb.cpu().numpy() - ob)) <= tolphi
    return Qg


def test_config1_fp64(B, oracle):
    cfg = inputs.config1()
    g, o = _pair(B, oracle, cfg)
    _cmp_solve(g, o, 1e-11, 1e-9, False)
    for j in (1, 2, 33, cfg.Ns):
        assert np.max(np.abs(g.get_slice(0, j).cpu().numpy() - o.get_slice(0, j))) < 1e-9, j


def test_config1_fp32(B, oracle):
    cfg = inputs.config1()
    g, o = _pair(B, oracle, cfg, precision="f32")
    g.propagate(); o.propagate()
    Qg, pa, _ = g.density_operators()
    Qo, oa, _ = o.density_operators()
    assert abs(Qg - Qo) < 2e-4 * abs(Qo)
    assert np.max(np.abs(pa.cpu().numpy() - oa)) < 2e-4 * np.max(np.abs(oa))


@pytest.mark.parametrize("grid", [(8, 16, 32), (32, 8, 16), (16, 64, 8), (64, 32, 16), (8, 32, 32), (64, 16, 16), (16, 64, 64), (1, 32, 32)])
@pytest.mark.parametrize("precision", ["f64", "f32"])
def test_ragged_diblock_complex_fields(B, oracle, grid, precision):
    """Anisotropic grids: every pencil length 8..64 appears along every dimension; complex (CL-like) fields.  The last four
    have square yz-planes (the fused plane kernel) under an x dimension of a different length."""
    cfg = inputs.small_diblock(grid=grid, cell=(3.0, 4.0, 5.0), Ns=10, fA=0.4)
    g, o = _pair(B, oracle, cfg, precision=precision)
    if precision == "f64":
        _cmp_solve(g, o, 1e-11, 1e-9, True)
        for which, j in ((0, 1), (0, 10), (1, 1), (1, 7), (1, 10)):
            assert np.max(np.abs(g.get_slice(which, j).cpu().numpy() - o.get_slice(which, j))) < 1e-9, (which, j)
    else:
        g.propagate(); o.propagate()
        Qg, pa, pb = g.density_operators()
        Qo, oa, ob = o.density_operators()
        assert abs(Qg - Qo) < 2e-4 * abs(Qo)
        assert np.max(np.abs(pa.cpu().numpy() - oa)) < 2e-4 and np.max(np.abs(pb.cpu().numpy() - ob)) < 2e-4


@pytest.mark.parametrize("n", [128, 256])
def test_long_pencils_truncated_march(B, oracle, n):
    """Pencil lengths 128 and 256 along each dimension in turn (the other two short), 4 contour steps."""
    for perm in range(3):
        grid = [8, 8, 16]; grid[perm] = n
        cfg = inputs.small_diblock(grid=tuple(grid), cell=(3.0, 4.0, 5.0), Ns=10, fA=0.4, seed=perm)
        g, o = _pair(B, oracle, cfg)
        g.propagate(4); o.propagate(4)
        for which in (0, 1):
            assert np.max(np.abs(g.get_slice(which, 4).cpu().numpy() - o.get_slice(which, 4))) < 1e-10, (grid, which)


def test_uniform_field_and_invariants_on_device(B):
    """Device-only properties that hold at any size: uniform field closed form; mean q_j q+_{Ns-j} = Q; mean phi."""
    grid, Ns = (32, 32, 32), 20
    g = B.Fts(grid, (4.0, 4.0, 4.0), Ns, "external")
    w0 = 0.3 - 1.1j
    g.set_fields(torch.full(grid, w0, dtype=torch.complex128, device="cuda:0"))
    g.propagate()
    Q, phi, _ = g.density_operators()
    assert abs(Q - np.exp(-w0)) < 1e-13 and float((phi - 1).abs().max()) < 1e-12
    cfg = inputs.small_diblock(grid=(32, 32, 32), Ns=20, fA=0.4)
    g = B.Fts(cfg.grid, cfg.cell, cfg.Ns, "diblock", store_both=1, **_kw(cfg))
    g.set_fields(_dev(cfg.f0), _dev(cfg.f1))
    g.propagate()
    Q, pa, pb = g.density_operators()
    for j in range(0, Ns + 1, 3):
        Qj = complex((g.get_slice(0, j) * g.get_slice(1, Ns - j)).mean().item())
        assert abs(Qj - Q) < 1e-12 * abs(Q)
    assert abs(complex(pa.mean().item()) - cfg.fA) < 1e-12 and abs(complex((pa + pb).mean().item()) - 1) < 1e-12


def test_philox_normals_match_oracle(B, oracle):
    z = B.debug_normals(12345678901234, 7, 1, 2 ** 33 + 5, 4096).cpu().numpy()
    ref = np.array([oracle.normal(12345678901234, 7, 1, 2 ** 33 + 5 + i) for i in range(4096)])
    assert np.max(np.abs(z - ref)) < 1e-13          # same Philox integers; libm vs CUDA log/cos differ by ulps


def test_philox_words_bit_identical_over_a_million_counters(B, oracle):
    """the device's and the oracle's Philox4x32-10 outputs are the same integers, for 2^20 counters: consecutive
    sites across the 2^32 boundary of the site index, a step index with a high word, both field ids."""
    import ctypes as C
    n = 1 << 19
    olib = oracle.lib()
    c, k, o = (C.c_uint32 * 4)(), (C.c_uint32 * 2)(), (C.c_uint32 * 4)()
    for seed, step, field, site0 in ((0x0123456789ABCDEF, 7, 0, 2 ** 32 - n // 2), (42, 2 ** 35 + 3, 1, 0)):
        dev = B.debug_philox(seed, step, field, site0, n).cpu().numpy()
        ref = np.empty((n, 4), np.int64)
        k[0], k[1] = seed & 0xFFFFFFFF, seed >> 32
        c[2], c[3] = step & 0xFFFFFFFF, field ^ (((step >> 32) << 8) & 0xFFFFFFFF)
        for i in range(n):
            site = site0 + i
            c[0], c[1] = site & 0xFFFFFFFF, site >> 32
            olib.oracle_philox4x32_10(c, k, o)
            ref[i, 0], ref[i, 1], ref[i, 2], ref[i, 3] = o[0], o[1], o[2], o[3]
        assert np.array_equal(dev, ref)


@pytest.mark.parametrize("seidel", [0, 1])
def test_scft_trajectory(B, oracle, seidel):
    cfg = inputs.config2(grid=(16, 16, 16), Ns=20)
    cfg.fA = 0.3
    g, o = _pair(B, oracle, cfg)
    for it in range(5):
        Hg, rg = g.scft_step(5.0, 5.0, seidel)
        Ho, ro = o.scft_step(5.0, 5.0, seidel)
        assert abs(Hg - Ho) < 1e-10 and abs(rg[0] - ro[0]) < 1e-9 and abs(rg[1] - ro[1]) < 1e-9, it
    a, b = g.get_fields(); oa, ob = o.get_fields()
    assert np.max(np.abs(a.cpu().numpy() - oa)) < 1e-9 and np.max(np.abs(b.cpu().numpy() - ob)) < 1e-9


@pytest.mark.parametrize("model,scheme", [("diblock", 0), ("diblock", 1), ("edwards", 0), ("edwards", 1)])
def test_cl_trajectory_10_steps(B, oracle, model, scheme):
    """Identical Philox noise on both sides: fields agree to 1e-8 after 10 steps (north_star)."""
    if model == "diblock":
        cfg = inputs.small_diblock(grid=(16, 16, 16), cell=(4.0, 4.0, 4.0), Ns=10, fA=0.4, C=20.0, complex_fields=False)
    else:
        cfg = inputs.config4(grid=(16, 16, 16), cell=(4.0, 4.0, 4.0), Ns=10)
    g, o = _pair(B, oracle, cfg)
    for step in range(10):
        g.cl_step(0.01, scheme, 2024, step)
        o.cl_step(0.01, scheme, 2024, step)
    a, b = g.get_fields(); oa, ob = o.get_fields()
    assert np.max(np.abs(a.cpu().numpy() - oa)) < 1e-8
    if model == "diblock":
        assert np.max(np.abs(b.cpu().numpy() - ob)) < 1e-8
    assert np.max(np.abs(a.cpu().numpy() - cfg.f0)) > 1e-3      # the fields did move


@pytest.mark.parametrize("model", ["edwards", "diblock", "external"])
def test_operators(B, oracle, model):
    if model == "diblock":
        cfg = inputs.small_diblock(grid=(16, 16, 16), Ns=10, fA=0.4)
    elif model == "edwards":
        cfg = inputs.config4(grid=(16, 16, 16), cell=(4.0, 4.0, 4.0), Ns=10)
    else:
        cfg = inputs.config1(Ns=16)
    g, o = _pair(B, oracle, cfg)
    g.propagate(); o.propagate()
    g.density_operators(); o.density_operators()
    for x, y in zip(g.operators(), o.operators()):
        assert abs(x - y) < 1e-9 * max(1.0, abs(y))


def test_error_codes(B):
    g = B.Fts((16, 16, 16), (4.0,) * 3, 10, "external")
    with pytest.raises(B.FtsError) as e:
        g.propagate()
    assert e.value.status == 2                         # fields not set
    g.set_fields(torch.zeros((16, 16, 16), dtype=torch.complex128, device="cuda:0"))
    with pytest.raises(B.FtsError) as e:
        g.density_operators()
    assert e.value.status == 2                         # density before propagate
    with pytest.raises(B.FtsError) as e:
        g.cl_step(0.01, 0, 1, 0)
    assert e.value.status == 6
    g.set_fields(torch.full((16, 16, 16), float("nan"), dtype=torch.complex128, device="cuda:0"))
    g.propagate()
    with pytest.raises(B.FtsError) as e:
        g.density_operators()
    assert e.value.status == 5                         # FTS_ENONFINITE


def test_determinism(B):
    cfg = inputs.small_diblock(grid=(32, 16, 16), Ns=10, fA=0.4)
    outs = []
    for _ in range(2):
        g = B.Fts(cfg.grid, cfg.cell, cfg.Ns, "diblock", **_kw(cfg))
        g.set_fields(_dev(cfg.f0), _dev(cfg.f1))
        g.cl_step(0.01, 0, 5, 0)
        g.propagate()
        Q, pa, pb = g.density_operators()
        outs.append((Q, pa.clone(), pb.clone()))
    assert outs[0][0] == outs[1][0] and torch.equal(outs[0][1], outs[1][1]) and torch.equal(outs[0][2], outs[1][2])


# ------------------------------------------------------------------------------------------------
# the march schedules (persistent ticket kernel with L2 slabs, stream-ordered launches) and full-size runs
# ------------------------------------------------------------------------------------------------
@pytest.mark.parametrize("opts", [{}, {"march": 1}, {"march": 1, "plane": 0}, {"march": 1, "tline": 0}, {"march": 1, "plane": 0, "graph": 0, "tline": 0}, {"march": 2}, {"march": 2, "slab_bytes": 65536},
                                  {"march": 2, "slab_bytes": 32768, "lag": 3}, {"march": 2, "interleave": 0, "slab_bytes": 131072}, {"march": 2, "tz": 8}])
@pytest.mark.parametrize("precision", ["f64", "f32"])
def test_march_schedules_agree(B, oracle, opts, precision):
    """Cubic 32^3 grid: the automatic choice (graph-replayed launches with the fused yz-plane kernel), the per-phase launches
    with and without plane fusion and graph, the persistent ticket kernel with one slab, 8 and 16 slabs and different pipeline
    lags all reproduce the oracle; they are also bit-identical to each other (fts_set_option)."""
    cfg = inputs.small_diblock(grid=(32, 32, 32), cell=(4.0, 4.0, 4.0), Ns=10, fA=0.4)
    ref, _ = _pair(B, oracle, cfg, precision=precision)
    ref.propagate()
    Qr, par, pbr = ref.density_operators()
    g, o = _pair(B, oracle, cfg, precision=precision)
    for k, v in opts.items():
        g.set_option(k, v)
    g.set_fields(*[torch.from_numpy(np.ascontiguousarray(f)).to("cuda:0").to(g.cdtype) for f in (cfg.f0, cfg.f1)])
    g.propagate(); o.propagate()
    Qg, pa, pb = g.density_operators()
    Qo, oa, ob = o.density_operators()
    tol = (1e-11, 1e-9) if precision == "f64" else (2e-4, 2e-4)
    assert abs(Qg - Qo) <= tol[0] * abs(Qo)
    assert np.max(np.abs(pa.cpu().numpy() - oa)) <= tol[1] and np.max(np.abs(pb.cpu().numpy() - ob)) <= tol[1]
    assert Qg == Qr and torch.equal(pa, par) and torch.equal(pb, pbr)      # the schedule does not change the arithmetic


def test_set_option_rejects_bad_values(B):
    g = B.Fts((16, 16, 16), (4.0,) * 3, 8, "external")
    for key, val in (("nonsense", 1), ("march", 7), ("tz", 5), ("lag", 1000)):
        with pytest.raises(B.FtsError) as e:
            g.set_option(key, val)
        assert e.value.status == 1                     # FTS_EINVAL
    with pytest.raises(B.FtsError) as e:
        g.set_option("march", 3)                       # the TMA march needs a cubic 128^3 or 256^3 grid
    assert e.value.status == 6                         # FTS_EUNSUPPORTED


@pytest.mark.parametrize("precision", ["f64"])
@pytest.mark.parametrize("model,nsteps", [("diblock", 6), ("diblock", 1), ("external", 4)])
def test_tma_march_equals_ticket_march_128(B, precision, model, nsteps):
    """128^3: the TMA march (fts_march2.cuh, automatic choice) and the ticket march (fts_march.cuh) use the same butterflies;
    the TMA march runs its inverse transform as conj o forward o conj, so the two agree to rounding on every slice, including
    across the block junction.  (Oracle parity of this size: test_full_size_*.)"""
    Ns = 8
    if model == "diblock":
        cfg = inputs.small_diblock(grid=(128, 128, 128), cell=(9.0, 10.0, 11.0), Ns=Ns, fA=0.5)
        kw = dict(fA=cfg.fA, chiN=cfg.chiN, Cc=cfg.C)
        fields = (cfg.f0, cfg.f1)
    else:
        rng = np.random.default_rng(11)
        fields = ((0.4 + 0.3 * rng.normal(size=(128,) * 3) + 0.2j * rng.normal(size=(128,) * 3)).astype(np.complex128),)
        kw = {}
    outs = []
    for mode in (2, 3):
        g = B.Fts((128,) * 3, (9.0, 10.0, 11.0), Ns, model, precision=precision, options={"march": mode}, store_both=1, **kw)
        g.set_fields(*[torch.from_numpy(np.ascontiguousarray(f)).to("cuda:0").to(g.cdtype) for f in fields])
        g.propagate(nsteps)
        sl = [g.get_slice(w, j).clone() for w in ((0, 1) if model == "diblock" else (0,)) for j in range(nsteps + 1)]
        outs.append(sl)
        del g
    for a, b in zip(*outs):
        assert (a - b).abs().max().item() < 1e-13


def test_zero_and_one_step_march(B, oracle):
    """Degenerate marches: 0 steps leaves q_0 = q+_0 = 1 and Q = 1; 1 step equals one Eq. 12 application of the oracle."""
    cfg = inputs.small_diblock(grid=(16, 16, 16), cell=(4.0, 4.0, 4.0), Ns=10, fA=0.4)
    g, o = _pair(B, oracle, cfg)
    g.propagate(0)
    for which in (0, 1):
        assert torch.equal(g.get_slice(which, 0), torch.ones(cfg.grid, dtype=torch.complex128, device="cuda:0"))
    g.propagate(1); o.propagate(1)
    for which in (0, 1):
        assert np.max(np.abs(g.get_slice(which, 1).cpu().numpy() - o.get_slice(which, 1))) < 1e-12
    with pytest.raises(B.FtsError) as e:
        g.density_operators()                          # a truncated march has no densities
    assert e.value.status == 2


@pytest.mark.parametrize("model", ["edwards", "external"])
def test_single_propagator_cubic_64(B, oracle, model):
    """One propagator (q+ = q) through the persistent kernel at 64^3: T and U phases alternate with no second propagator."""
    if model == "edwards":
        cfg = inputs.config4(Ns=10)
    else:
        cfg = inputs.config1(grid=(64, 64, 64), cell=(8.0, 8.0, 8.0), Ns=10)
    g, o = _pair(B, oracle, cfg)
    _cmp_solve(g, o, 1e-11, 1e-9, False)
    assert np.max(np.abs(g.get_slice(0, cfg.Ns).cpu().numpy() - o.get_slice(0, cfg.Ns))) < 1e-9


CL_SEED = 20120454


@pytest.fixture(scope="module")
def oracle_cfg5s(oracle):
    """Config 5s (128^3, Ns = 100, q and q+: 200 RQM4 steps) on the oracle, ONCE per session (~3 x 110 s + 40 s on one core): a
    full solve (Q, phi_A, phi_B, operators) and the complex-Langevin step from the same fields in both schemes (each solves again)."""
    cfg = inputs.config5(128)
    o = oracle.Oracle(cfg.grid, cfg.cell, cfg.Ns, cfg.model, precision="f64", **_kw(cfg))
    o.set_fields(cfg.f0, cfg.f1)
    o.propagate()
    Q, pa, pb = o.density_operators()
    qN = o.get_slice(0, cfg.Ns)
    ops = o.operators()                                # H, mu, Pi out of the same solve (Pi: 101 Laplacians, ~40 s)
    o.cl_step(cfg.dt, 0, CL_SEED, 0)
    wp, wm = o.get_fields()
    o.set_fields(cfg.f0, cfg.f1)
    o.cl_step(cfg.dt, 1, CL_SEED, 0)                    # the semi-implicit update of Eq. 10-11 from the same fields (one more solve)
    si = o.get_fields()
    del o
    return cfg, Q, pa, pb, qN, wp, wm, ops, si


@pytest.mark.parametrize("precision", ["f64", "f32"])
def test_config5s_full_oracle_solve_and_cl_step(B, oracle_cfg5s, precision):
    """SURVEY 8(d), config 5s through the TMA march in BOTH slice stores - the library default (meet-in-the-middle, densities
    fused into the march) and the full store bench.py times by default (store_both = 1, densities by density_store_kernel):
    Q to 1e-11 (2e-4 in complex64), phi_A, phi_B and q(r,1) element-wise to 1e-9 (2e-4), the fields after one fts_cl_step with
    identical Philox noise to 1e-9 (2e-4), and - N2 at scale, full store - H, mu and Pi over the 2 x 101 stored slices of 128^3
    and one semi-implicit step (Eq. 10-11, scheme 1), all against the oracle's full 200-step solves."""
    cfg, Qo, oa, ob, qN, wpo, wmo, ops_o, si_o = oracle_cfg5s
    dt = torch.complex128 if precision == "f64" else torch.complex64
    tq, tp = (1e-11, 1e-9) if precision == "f64" else (2e-4, 2e-4)
    g = B.Fts(cfg.grid, cfg.cell, cfg.Ns, cfg.model, precision=precision, **_kw(cfg))
    g.set_fields(_dev(cfg.f0, dt), _dev(cfg.f1, dt))
    g.propagate()
    Qg, pa, pb = g.density_operators()
    assert abs(Qg - Qo) <= tq * abs(Qo), (Qg, Qo)
    assert np.max(np.abs(pa.cpu().numpy() - oa)) <= tp and np.max(np.abs(pb.cpu().numpy() - ob)) <= tp
    assert np.max(np.abs(g.get_slice(0, cfg.Ns).cpu().numpy() - qN)) <= tp * max(1.0, np.max(np.abs(qN)))
    g.cl_step(cfg.dt, 0, CL_SEED, 0)
    wp, wm = g.get_fields()
    assert np.max(np.abs(wp.cpu().numpy() - wpo)) <= tp * max(1.0, np.max(np.abs(wpo)))
    assert np.max(np.abs(wm.cpu().numpy() - wmo)) <= tp * max(1.0, np.max(np.abs(wmo)))
    g.close(); del g
    f = B.Fts(cfg.grid, cfg.cell, cfg.Ns, cfg.model, precision=precision, store_both=1, **_kw(cfg))      # bench.py --store full
    f.set_fields(_dev(cfg.f0, dt), _dev(cfg.f1, dt))
    f.propagate()
    Qf, fa, fb = f.density_operators()
    assert abs(Qf - Qo) <= tq * abs(Qo), (Qf, Qo)
    assert np.max(np.abs(fa.cpu().numpy() - oa)) <= tp and np.max(np.abs(fb.cpu().numpy() - ob)) <= tp
    for k, (x, y) in enumerate(zip(f.operators(), ops_o)):      # H/(CV), mu = ln C - ln Q, Pi (reading A-14)
        tol = 1e-9 if precision == "f64" else (2e-4 if k < 2 else 5e-3)      # complex64 Pi: -k^2 amplifies the rounding of 101 slices
        assert abs(x - y) <= tol * max(1.0, abs(y)), (k, x, y)
    f.cl_step(cfg.dt, 0, CL_SEED, 0)
    wp, wm = f.get_fields()
    assert np.max(np.abs(wp.cpu().numpy() - wpo)) <= tp * max(1.0, np.max(np.abs(wpo)))
    assert np.max(np.abs(wm.cpu().numpy() - wmo)) <= tp * max(1.0, np.max(np.abs(wmo)))
    f.set_fields(_dev(cfg.f0, dt), _dev(cfg.f1, dt))    # N2 at scale: Eq. 10-11 (scheme 1; filter passes at pencil length 128) from the same fields
    f.cl_step(cfg.dt, 1, CL_SEED, 0)
    for x, y in zip(f.get_fields(), si_o):
        assert np.max(np.abs(x.cpu().numpy() - y)) <= tp * max(1.0, np.max(np.abs(y)))


@pytest.fixture(scope="module")
def oracle_cfg5_first8(oracle):
    """Config 5 (256^3): the first 8 contour steps of q and q+ on the oracle (16 RQM4 steps of 2^24 points, ~100 s), once."""
    cfg = inputs.config5(256)
    o = oracle.Oracle(cfg.grid, cfg.cell, cfg.Ns, cfg.model, precision="f64", **_kw(cfg))
    o.set_fields(cfg.f0, cfg.f1)
    o.propagate(8)
    sl = {(w, j): o.get_slice(w, j) for w in (0, 1) for j in (1, 8)}
    del o
    return cfg, sl


@pytest.mark.parametrize("precision", ["f64", "f32"])
def test_config5_truncated_march_and_invariants(B, oracle_cfg5_first8, precision):
    """Config 5 (256^3) in the launch configuration bench.py times: slices 1 and 8 of both propagators against the oracle
    (first 8 steps), then properties that hold at any size on the full march with every slice kept."""
    cfg, sl = oracle_cfg5_first8
    dt = torch.complex128 if precision == "f64" else torch.complex64
    g = B.Fts(cfg.grid, cfg.cell, cfg.Ns, cfg.model, precision=precision, store_both=1, **_kw(cfg))
    g.set_fields(_dev(cfg.f0, dt), _dev(cfg.f1, dt))
    g.propagate(8)
    tol = 1e-10 if precision == "f64" else 2e-4
    for (which, j), ref in sl.items():
        assert np.max(np.abs(g.get_slice(which, j).cpu().numpy() - ref)) <= tol * max(1.0, np.max(np.abs(ref))), (which, j)
    g.propagate()
    Q, pa, pb = g.density_operators()
    rel = 1e-11 if precision == "f64" else 2e-4
    for j in (0, 1, 37, 50, 99, 100):
        Qj = complex((g.get_slice(0, j).to(torch.complex128) * g.get_slice(1, cfg.Ns - j).to(torch.complex128)).mean().item())
        assert abs(Qj - Q) <= rel * abs(Q), j
    assert abs(complex(pa.to(torch.complex128).mean().item()) - cfg.fA) <= rel
    assert abs(complex((pa + pb).to(torch.complex128).mean().item()) - 1.0) <= rel
    # the default (meet-in-the-middle) store, densities accumulated inside the march, gives the same Q bit for bit and the same
    # densities to rounding (the full store is summed in one pass with fp64 accumulators, in a different order)
    del g
    g2 = B.Fts(cfg.grid, cfg.cell, cfg.Ns, cfg.model, precision=precision, **_kw(cfg))
    g2.set_fields(_dev(cfg.f0, dt), _dev(cfg.f1, dt))
    g2.propagate()
    Q2, pa2, pb2 = g2.density_operators()
    assert Q2 == Q
    assert float((pa2 - pa).abs().max()) <= (1e-13 if precision == "f64" else 1e-5) and float((pb2 - pb).abs().max()) <= (1e-13 if precision == "f64" else 1e-5)


# ------------------------------------------------------------------------------------------------
# BASELINE configs 2-4 at full size: trajectory parity over the first iterations; parity of one solve at seeded
# "developed" fields (inputs.developed: nothing the CUDA path produced is ever fed to the oracle); and properties that
# hold at any size after a long GPU run (the oracle is too slow for 200-1000 iterations)
# ------------------------------------------------------------------------------------------------
def _developed_solve_parity(B, oracle, cfg, precision="f64", tolQ=1e-11, tolphi=1e-9, operators=False, real_fields=False):
    f0, f1 = inputs.developed(cfg)
    dt = torch.complex128 if precision == "f64" else torch.complex64
    g = B.Fts(cfg.grid, cfg.cell, cfg.Ns, cfg.model, precision=precision, store_both=1 if operators else 0, **_kw(cfg))
    if real_fields:                                    # the real parts of the developed fields, marched packed (z = q + i q+)
        f0, f1 = np.ascontiguousarray(f0.real).astype(np.complex128), np.ascontiguousarray(f1.real).astype(np.complex128)
        g.set_option("real_fields", 1)
    o = oracle.Oracle(cfg.grid, cfg.cell, cfg.Ns, cfg.model, precision="f64", **_kw(cfg))
    g.set_fields(_dev(f0, dt), None if f1 is None else _dev(f1, dt))
    o.set_fields(f0, f1)
    g.propagate(); o.propagate()
    Qg, pa, pb = g.density_operators()
    Qo, oa, ob = o.density_operators()
    assert np.isfinite(Qg.real) and abs(Qg - Qo) <= tolQ * abs(Qo), (Qg, Qo)
    assert np.max(np.abs(pa.cpu().numpy() - oa)) <= tolphi
    if ob is not None:
        assert np.max(np.abs(pb.cpu().numpy() - ob)) <= tolphi
    if operators:
        for x, y in zip(g.operators(), o.operators()):     # H (Eq. 2), mu = ln C - ln Q, Pi (reading A-14)
            assert abs(x - y) < 1e-9 * max(1.0, abs(y))


def _invariants(g, cfg, rel):
    g.propagate()
    Q, pa, pb = g.density_operators()
    assert np.isfinite(Q.real) and np.isfinite(Q.imag)
    two = cfg.model == "diblock"
    for j in (0, cfg.Ns // 3, cfg.Ns):
        Qj = complex((g.get_slice(0, j).to(torch.complex128) * g.get_slice(1, cfg.Ns - j).to(torch.complex128)).mean().item())
        assert abs(Qj - Q) <= rel * abs(Q), j
    tot = pa + pb if two else pa
    assert abs(complex(tot.to(torch.complex128).mean().item()) - 1.0) <= rel
    if two:
        assert abs(complex(pa.to(torch.complex128).mean().item()) - cfg.fA) <= rel


def test_config2_scft_full_size(B, oracle):
    """32^3, Ns = 100, fA = 0.3, chiN = 20, Seidel: 4 iterations side by side with the oracle; all 200 iterations on the
    GPU (residual falls, invariants hold); one solve at developed fields against the oracle."""
    cfg = inputs.config2()
    g, o = _pair(B, oracle, cfg)
    gr, _ = _pair(B, oracle, cfg, store_both=0)         # as bench.py runs SCFT workloads: real_fields = 1, q and q+ packed, Ns = 100, jA = 30
    gr.set_option("real_fields", 1)
    for it in range(4):
        Hg, rg = g.scft_step(*cfg.dt_scft, 1)
        Hr, rr = gr.scft_step(*cfg.dt_scft, 1)
        Ho, ro = o.scft_step(*cfg.dt_scft, 1)
        assert abs(Hg - Ho) < 1e-10 and abs(rg[0] - ro[0]) < 1e-9 and abs(rg[1] - ro[1]) < 1e-9, it
        assert abs(Hr - Ho) < 1e-10 and abs(rr[0] - ro[0]) < 1e-9 and abs(rr[1] - ro[1]) < 1e-9, it
    for x, y in zip(gr.get_fields(), o.get_fields()):
        assert np.max(np.abs(x.cpu().numpy() - y)) < 1e-9
    _developed_solve_parity(B, oracle, cfg, real_fields=True)
    res = []
    for it in range(4, cfg.iters):
        H, r = g.scft_step(*cfg.dt_scft, 1)
        res.append(max(r))
    assert res[-1] < res[0]                            # the relaxation makes progress
    _invariants(g, cfg, 1e-11)
    _developed_solve_parity(B, oracle, cfg)
    _developed_solve_parity(B, oracle, cfg, precision="f32", tolQ=2e-4, tolphi=2e-4)      # complex64 at full size


@pytest.mark.parametrize("precision", ["f64", "f32"])
def test_config3_scft_full_size(B, oracle, precision):
    """64^3, Ns = 200 (jA = 70), q+ batched with q: 30 Seidel iterations on the GPU (invariants), one solve at developed
    fields against the oracle."""
    cfg = inputs.config3()
    g, o = _pair(B, oracle, cfg, precision=precision)
    if precision == "f64":                             # one Seidel iteration side by side (2 x 400 RQM4 steps on the oracle, ~75 s)
        gr, _ = _pair(B, oracle, cfg, store_both=0)     # ... and the same iteration as bench.py runs it: real_fields = 1 (packed march, Ns = 200, jA = 70)
        gr.set_option("real_fields", 1)
        Hg, rg = g.scft_step(*cfg.dt_scft, 1)
        Hr, rr = gr.scft_step(*cfg.dt_scft, 1)
        Ho, ro = o.scft_step(*cfg.dt_scft, 1)
        assert abs(Hg - Ho) < 1e-10 and abs(rg[0] - ro[0]) < 1e-9 and abs(rg[1] - ro[1]) < 1e-9
        assert abs(Hr - Ho) < 1e-10 and abs(rr[0] - ro[0]) < 1e-9 and abs(rr[1] - ro[1]) < 1e-9
        for x, y in zip(g.get_fields(), o.get_fields()):
            assert np.max(np.abs(x.cpu().numpy() - y)) < 1e-9
        for x, y in zip(gr.get_fields(), o.get_fields()):
            assert np.max(np.abs(x.cpu().numpy() - y)) < 1e-9
        gr.close(); del gr
    del o
    for it in range(30):
        H, r = g.scft_step(*cfg.dt_scft, 1)
    assert np.isfinite(H.real) and max(r) < 1.0
    _invariants(g, cfg, 1e-11 if precision == "f64" else 2e-4)
    if precision == "f64":
        _developed_solve_parity(B, oracle, cfg)
        _developed_solve_parity(B, oracle, cfg, real_fields=True)      # the packed march at developed (real) fields, ~40 s of oracle
    else:
        _developed_solve_parity(B, oracle, cfg, precision="f32", tolQ=2e-4, tolphi=2e-4)


def test_config4_edwards_cl_full_size(B, oracle):
    """64^3 Edwards solution, B = 1, C = 10, dt = 0.01: north_star's criterion at the config's own size - 10 CL steps side by
    side with identical Philox noise, fields within 1e-8 (~95 s of oracle); 100 more steps on the GPU (invariants); one solve
    plus the operators H, mu, Pi at developed fields against the oracle."""
    cfg = inputs.config4()
    g, o = _pair(B, oracle, cfg)
    for step in range(10):
        g.cl_step(cfg.dt, 0, 4242, step); o.cl_step(cfg.dt, 0, 4242, step)
        if step == 1:
            assert np.max(np.abs(g.get_fields()[0].cpu().numpy() - o.get_fields()[0])) < 1e-9
    a, _ = g.get_fields(); oa, _ = o.get_fields()
    assert np.max(np.abs(a.cpu().numpy() - oa)) < 1e-8
    for step in range(10, 110):
        g.cl_step(cfg.dt, 0, 4242, step)
    _invariants(g, cfg, 1e-11)
    _developed_solve_parity(B, oracle, cfg, operators=True)
    _developed_solve_parity(B, oracle, cfg, precision="f32", tolQ=2e-4, tolphi=2e-4)      # complex64 at full size


@pytest.mark.parametrize("model", ["diblock", "edwards"])
def test_fp32_field_updates_track_the_fp64_oracle(B, oracle, model):
    """complex64 mode through the update kernels: 5 CL steps (identical Philox noise, rounded to float) and, for the
    diblock, 3 SCFT iterations stay within the fp32 tolerance of north_star (2e-4 relative) of the fp64 oracle."""
    if model == "diblock":
        cfg = inputs.small_diblock(grid=(16, 16, 16), cell=(4.0, 4.0, 4.0), Ns=10, fA=0.4, C=20.0, complex_fields=False)
    else:
        cfg = inputs.config4(grid=(16, 16, 16), cell=(4.0, 4.0, 4.0), Ns=10)
    g, o = _pair(B, oracle, cfg, precision="f32")
    for step in range(5):
        g.cl_step(0.01, 0, 77, step); o.cl_step(0.01, 0, 77, step)
    a, b = g.get_fields(); oa, ob = o.get_fields()
    assert np.max(np.abs(a.cpu().numpy() - oa)) < 2e-4 * max(1.0, np.max(np.abs(oa)))
    if model == "diblock":
        assert np.max(np.abs(b.cpu().numpy() - ob)) < 2e-4 * max(1.0, np.max(np.abs(ob)))
        cfg2 = inputs.config2(grid=(16, 16, 16), Ns=20)
        g2, o2 = _pair(B, oracle, cfg2, precision="f32")
        for it in range(3):
            Hg, rg = g2.scft_step(5.0, 5.0, 1)
            Ho, ro = o2.scft_step(5.0, 5.0, 1)
            assert abs(Hg - Ho) < 2e-4 * max(1.0, abs(Ho)) and abs(rg[0] - ro[0]) < 2e-4 and abs(rg[1] - ro[1]) < 2e-4 * max(1.0, ro[1]), it


@pytest.mark.parametrize("n,precision,reps", [(16, "f64", 500), (32, "f64", 1000), (64, "f64", 300), (64, "f32", 300), (128, "f64", 60), (128, "f32", 60), (256, "f64", 6)])
def test_march_soak_bit_identical(B, n, precision, reps):
    """The dependency protocol under changing timing: repeated solves of the same fields (persistent kernel, work items
    claimed dynamically by ~300-450 CTAs) must be bit-identical every time; a race would show as a differing bit."""
    cfg = inputs.small_diblock(grid=(n, n, n), cell=(4.0, 4.0, 4.0), Ns=10, fA=0.4)
    dt = torch.complex128 if precision == "f64" else torch.complex64
    g = B.Fts(cfg.grid, cfg.cell, cfg.Ns, "diblock", precision=precision, store_both=n % 64 == 0, **_kw(cfg))      # both store layouts
    g.set_fields(_dev(cfg.f0, dt), _dev(cfg.f1, dt))
    g.propagate()
    Q0, pa0, pb0 = g.density_operators()
    pa0, pb0 = pa0.clone(), pb0.clone()
    last = g.get_slice(1, cfg.Ns).clone()
    for rep in range(reps):
        if rep % 3 == 1:
            torch.empty(64 << 20, dtype=torch.uint8, device="cuda:0").zero_()      # perturb L2 / timing
        g.propagate()
        Q, pa, pb = g.density_operators()
        assert Q == Q0 and torch.equal(pa, pa0) and torch.equal(pb, pb0), rep
        assert torch.equal(g.get_slice(1, cfg.Ns), last), rep


# ------------------------------------------------------------------------------------------------
# S6: densities accumulated inside the march, meet-in-the-middle store (the default, store_both = 0)
# ------------------------------------------------------------------------------------------------
@pytest.mark.parametrize("model,grid,Ns,fA", [("diblock", (16, 16, 16), 20, 0.3), ("diblock", (32, 32, 32), 10, 0.4), ("diblock", (16, 8, 32), 12, 0.5),
                                               ("edwards", (16, 16, 16), 10, 0.5), ("external", (32, 32, 32), 6, 0.5), ("external", (8, 16, 8), 2, 0.5)])
@pytest.mark.parametrize("precision", ["f64", "f32"])
def test_meet_in_the_middle_store(B, oracle, model, grid, Ns, fA, precision):
    """Default store: Q and phi as with the full store and as the oracle's plain sum over all slices (block junction left, right
    and at the middle; one and two propagators; persistent and per-phase launches); retained slices 0..Ns/2 and Ns match the
    oracle; any other slice is FTS_ESTATE; Pi (needs every slice) is FTS_ESTATE."""
    if model == "diblock":
        cfg = inputs.small_diblock(grid=grid, cell=(3.0, 4.0, 5.0), Ns=Ns, fA=fA)
    elif model == "edwards":
        cfg = inputs.config4(grid=grid, cell=(4.0, 4.0, 4.0), Ns=Ns)
    else:
        cfg = inputs.config1(grid=grid, cell=(4.0, 4.0, 4.0), Ns=Ns)
    g, o = _pair(B, oracle, cfg, precision=precision, store_both=0)
    two = model == "diblock"
    if precision == "f64":
        _cmp_solve(g, o, 1e-11, 1e-9, two)
    else:
        g.propagate(); o.propagate()
        Qg, pa, pb = g.density_operators(); Qo, oa, ob = o.density_operators()
        assert abs(Qg - Qo) < 2e-4 * abs(Qo) and np.max(np.abs(pa.cpu().numpy() - oa)) < 2e-4 * max(1.0, np.max(np.abs(oa)))
        if two:
            assert np.max(np.abs(pb.cpu().numpy() - ob)) < 2e-4
    tol = 1e-9 if precision == "f64" else 2e-4
    for which in ((0, 1) if two else (0,)):
        for j in (0, 1, Ns // 2, Ns):
            assert np.max(np.abs(g.get_slice(which, j).cpu().numpy() - o.get_slice(which, j))) < tol, (which, j)
        if Ns // 2 + 1 < Ns:
            with pytest.raises(B.FtsError) as e:
                g.get_slice(which, Ns // 2 + 1)
            assert e.value.status == 2                 # FTS_ESTATE
    with pytest.raises(B.FtsError) as e:
        g.operators(want_pi=True)
    assert e.value.status == 2
    H, mu, _ = g.operators(want_pi=False)
    Ho, muo, _ = o.operators()
    assert abs(mu - muo) < (1e-10 if precision == "f64" else 2e-4) * max(1.0, abs(muo))
    # a truncated march keeps its last slice (the slice Q is taken from) and leaves the densities undefined
    k = Ns // 2 + 1 if Ns > 2 else 1
    g.propagate(k); o.propagate(k)
    assert np.max(np.abs(g.get_slice(0, k).cpu().numpy() - o.get_slice(0, k))) < tol
    with pytest.raises(B.FtsError):
        g.density_operators()


def test_workspace_halves_with_the_default_store(B):
    from paper_1204_5434_b200.binding import make_params, workspace_bytes
    a = workspace_bytes((64, 64, 64), 100, make_params("diblock", fA=0.5, store_both=0))
    b = workspace_bytes((64, 64, 64), 100, make_params("diblock", fA=0.5, store_both=1))
    field = 64 ** 3 * 16
    assert b - a == 2 * (101 - 52) * field            # Ns/2 + 2 slices per propagator instead of Ns + 1


# ------------------------------------------------------------------------------------------------
# N3: 1-D and 2-D grids (Fig. 1) as grids with dimensions of 1
# ------------------------------------------------------------------------------------------------
@pytest.mark.parametrize("grid,cell", [((64, 1, 1), (5.0, 1.0, 1.0)), ((1, 1, 128), (1.0, 1.0, 7.0)), ((1, 256, 1), (2.0, 9.0, 1.0)),
                                        ((32, 16, 1), (3.0, 4.0, 1.0)), ((1, 8, 64), (1.0, 3.0, 5.0)), ((128, 1, 8), (6.0, 1.0, 2.0))])
@pytest.mark.parametrize("precision", ["f64", "f32"])
def test_one_and_two_dimensional_grids(B, oracle, grid, cell, precision):
    """The same kernels with pencils of length 1 along the missing dimensions: propagator slices, Q, phi, one SCFT iteration
    (3-D filter passes of length 1) and one CL step (scheme 1: the Eq. 11 filter) against the oracle on the same grid."""
    cfg = inputs.small_diblock(grid=grid, cell=cell, Ns=12, fA=0.5, complex_fields=True)
    g, o = _pair(B, oracle, cfg, precision=precision)
    if precision == "f64":
        _cmp_solve(g, o, 1e-11, 1e-9, True)
        for which, j in ((0, 3), (1, 5), (0, 12), (1, 12)):
            assert np.max(np.abs(g.get_slice(which, j).cpu().numpy() - o.get_slice(which, j))) < 1e-9, (which, j)
        Hg, rg = g.scft_step(2.0, 2.0, 1); Ho, ro = o.scft_step(2.0, 2.0, 1)
        assert abs(Hg - Ho) < 1e-10 and abs(rg[0] - ro[0]) < 1e-9 and abs(rg[1] - ro[1]) < 1e-9
        g.cl_step(0.01, 1, 99, 0); o.cl_step(0.01, 1, 99, 0)
        for x, y in zip(g.get_fields(), o.get_fields()):
            assert np.max(np.abs(x.cpu().numpy() - y)) < 1e-9
    else:
        g.propagate(); o.propagate()
        Qg, pa, pb = g.density_operators(); Qo, oa, ob = o.density_operators()
        assert abs(Qg - Qo) < 2e-4 * abs(Qo)
        assert np.max(np.abs(pa.cpu().numpy() - oa)) < 2e-4 and np.max(np.abs(pb.cpu().numpy() - ob)) < 2e-4


@pytest.mark.parametrize("grid", [(256, 8, 8), (8, 128, 16), (16, 8, 256), (128, 16, 8)])
def test_filter_passes_at_long_pencils(B, oracle, grid):
    """pass_kernel (the 3-D filters of the SCFT / Eq. 11 updates and the Laplacian of Pi) at pencil lengths 128 and 256 along
    each dimension: one SCFT iteration, one semi-implicit CL step and the operators H, mu, Pi against the oracle."""
    cfg = inputs.small_diblock(grid=grid, cell=(7.0, 5.0, 6.0), Ns=8, fA=0.5)
    g, o = _pair(B, oracle, cfg)
    Hg, rg = g.scft_step(2.0, 2.0, 0); Ho, ro = o.scft_step(2.0, 2.0, 0)
    assert abs(Hg - Ho) < 1e-10 and abs(rg[0] - ro[0]) < 1e-9 and abs(rg[1] - ro[1]) < 1e-9
    g.cl_step(0.01, 1, 5, 3); o.cl_step(0.01, 1, 5, 3)
    for x, y in zip(g.get_fields(), o.get_fields()):
        assert np.max(np.abs(x.cpu().numpy() - y)) < 1e-9
    g.propagate(); o.propagate()
    for x, y in zip(g.operators(), o.operators()):
        assert abs(x - y) < 1e-9 * max(1.0, abs(y))


# ------------------------------------------------------------------------------------------------
# N1: real-field fast path (option "real_fields"): q and q+ marched together as z = q + i q+
# ------------------------------------------------------------------------------------------------
@pytest.mark.parametrize("grid,Ns,fA", [((16, 16, 16), 20, 0.3), ((32, 32, 32), 12, 0.5), ((8, 32, 16), 10, 0.8), ((64, 64, 64), 8, 0.25),
                                         ((128, 128, 128), 8, 0.5), ((1, 16, 64), 10, 0.4)])
@pytest.mark.parametrize("precision", ["f64", "f32"])
def test_real_fields_fast_path(B, oracle, grid, Ns, fA, precision):
    """Real W+ and W- (SCFT): the packed march reproduces the (complex) oracle: Q, phi_A, phi_B, slices of q and of q+ (block
    junction before, at and after the middle; ticket, per-phase-launch and TMA marches), both store layouts."""
    cfg = inputs.small_diblock(grid=grid, cell=(3.0, 4.0, 5.0), Ns=Ns, fA=fA, complex_fields=False)
    for store_both in (0, 1):
        g, o = _pair(B, oracle, cfg, precision=precision, store_both=store_both)
        g.set_option("real_fields", 1)
        g.propagate(); o.propagate()
        Qg, pa, pb = g.density_operators(); Qo, oa, ob = o.density_operators()
        tq, tp = (1e-11, 1e-9) if precision == "f64" else (2e-4, 2e-4)
        assert Qg.imag == 0.0 and abs(Qg - Qo) <= tq * abs(Qo), (Qg, Qo)
        assert np.max(np.abs(pa.cpu().numpy() - oa)) <= tp and np.max(np.abs(pb.cpu().numpy() - ob)) <= tp
        for which in (0, 1):
            for j in (0, 1, Ns // 2, Ns) + ((Ns - 1,) if store_both else ()):
                assert np.max(np.abs(g.get_slice(which, j).cpu().numpy() - o.get_slice(which, j))) <= tp, (which, j)
        with pytest.raises(B.FtsError) as e:
            g.cl_step(0.01, 0, 1, 0)
        assert e.value.status == 2
        g.set_option("real_fields", 0)                 # and back: the general path on the same context
        g.propagate()
        Q2, pa2, _ = g.density_operators()
        assert abs(Q2 - Qo) <= tq * abs(Qo) and np.max(np.abs(pa2.cpu().numpy() - oa)) <= tp


def test_real_fields_scft_trajectory_and_misuse(B, oracle):
    """SCFT iterations (both Seidel variants) with the option set follow the oracle; complex fields are reported (FTS_EINVAL);
    one-propagator models refuse the option (FTS_EUNSUPPORTED)."""
    cfg = inputs.config2(grid=(16, 16, 16), Ns=20)
    for seidel in (0, 1):
        g, o = _pair(B, oracle, cfg)
        g.set_option("real_fields", 1)
        for it in range(5):
            Hg, rg = g.scft_step(5.0, 5.0, seidel)
            Ho, ro = o.scft_step(5.0, 5.0, seidel)
            assert abs(Hg - Ho) < 1e-10 and abs(rg[0] - ro[0]) < 1e-9 and abs(rg[1] - ro[1]) < 1e-9, (seidel, it)
        for x, y in zip(g.get_fields(), o.get_fields()):
            assert np.max(np.abs(x.cpu().numpy() - y)) < 1e-9
    bad = inputs.small_diblock(grid=(16, 16, 16), Ns=10, fA=0.4, complex_fields=True)
    g, _ = _pair(B, oracle, bad)
    g.set_option("real_fields", 1)
    with pytest.raises(B.FtsError) as e:
        g.scft_step(1.0, 1.0, 0)
    assert e.value.status == 1                         # FTS_EINVAL: the declaration was wrong
    g1 = B.Fts((16, 16, 16), (4.0,) * 3, 8, "external")
    with pytest.raises(B.FtsError) as e:
        g1.set_option("real_fields", 1)
    assert e.value.status == 6


# ------------------------------------------------------------------------------------------------
# N3: linear multiblock chains (fts_set_blocks)
# ------------------------------------------------------------------------------------------------
@pytest.mark.parametrize("grid,Ns,blocks", [((16, 16, 16), 12, ([0, 1, 0], [2, 6, 4])), ((32, 32, 32), 16, ([1, 0, 1, 0], [2, 4, 6, 4])),
                                             ((8, 32, 16), 10, ([0, 1, 0], [4, 4, 2])), ((128, 128, 128), 8, ([0, 1, 0], [2, 4, 2])),
                                             ((64, 1, 1), 20, ([1, 0, 1], [6, 10, 4]))])
@pytest.mark.parametrize("store_both", [0, 1])
def test_multiblock_chains(B, oracle, grid, Ns, blocks, store_both):
    """ABA and ABAB chains through every march (ticket, per-phase launches, TMA), both store layouts, complex fields; then
    the real-field fast path on real fields; one SCFT iteration and one CL step follow the oracle with the same blocks."""
    fA = 0.5 if Ns % 4 == 0 else 0.4                   # the default diblock the context is created with must itself be valid
    cfg = inputs.small_diblock(grid=grid, cell=(3.0, 4.0, 5.0), Ns=Ns, fA=fA)
    g, o = _pair(B, oracle, cfg, store_both=store_both)
    g.set_blocks(*blocks); o.set_blocks(*blocks)
    _cmp_solve(g, o, 1e-11, 1e-9, True)
    for which in (0, 1):
        for j in (1, Ns // 2, Ns):
            assert np.max(np.abs(g.get_slice(which, j).cpu().numpy() - o.get_slice(which, j))) < 1e-9, (which, j)
    if grid[0] <= 32:
        Hg, rg = g.scft_step(2.0, 2.0, 1); Ho, ro = o.scft_step(2.0, 2.0, 1)
        assert abs(Hg - Ho) < 1e-10 and abs(rg[0] - ro[0]) < 1e-9 and abs(rg[1] - ro[1]) < 1e-9
        g.cl_step(0.01, 0, 3, 1); o.cl_step(0.01, 0, 3, 1)
        for x, y in zip(g.get_fields(), o.get_fields()):
            assert np.max(np.abs(x.cpu().numpy() - y)) < 1e-9
    real = inputs.small_diblock(grid=grid, cell=(3.0, 4.0, 5.0), Ns=Ns, fA=fA, complex_fields=False)
    g, o = _pair(B, oracle, real, store_both=store_both)
    g.set_blocks(*blocks); o.set_blocks(*blocks)
    g.set_option("real_fields", 1)
    _cmp_solve(g, o, 1e-11, 1e-9, True)
    with pytest.raises(B.FtsError) as e:
        g.set_blocks([0, 1], [3, Ns - 3])
    assert e.value.status == 1


@pytest.mark.parametrize("model", ["edwards", "diblock"])
def test_operators_of_the_cl_steps_entry_fields(B, oracle, model):
    """Config 4's deliverable is <mu>, <Pi> over a CL run: fts_operators after fts_cl_step reports the operators of the fields
    the step started from, out of the solve the step already did (no second solve).  Oracle: operators before its step."""
    if model == "edwards":
        cfg = inputs.config4(grid=(16, 16, 16), cell=(4.0, 4.0, 4.0), Ns=10)
    else:
        cfg = inputs.small_diblock(grid=(16, 16, 16), cell=(4.0, 4.0, 4.0), Ns=10, fA=0.4, C=20.0)
    g, o = _pair(B, oracle, cfg)
    n0 = B.launch_count()
    for step in range(3):
        o.propagate(); ref = o.operators()
        o.cl_step(0.01, 0, 5, step)
        g.cl_step(0.01, 0, 5, step)
        for x, y in zip(g.operators(), ref):
            assert abs(x - y) < 1e-9 * max(1.0, abs(y)), step
    with pytest.raises(B.FtsError):
        g.get_slice(0, 1)                              # the slices belong to the previous fields: not served
    g.propagate()
    o.propagate()
    for x, y in zip(g.operators(), o.operators()):
        assert abs(x - y) < 1e-9 * max(1.0, abs(y))


def test_streams_contexts_and_lifecycle(B, oracle):
    """Host-side robustness: work enqueued on a non-blocking side stream (the graph-replayed launch mode captures on a private
    stream and replays on the caller's), two contexts used alternately, and contexts created and destroyed repeatedly
    (graphs instantiated and released) all reproduce the default-stream result bit for bit."""
    cfg = inputs.small_diblock(grid=(32, 32, 32), cell=(4.0, 4.0, 4.0), Ns=10, fA=0.4)
    g, o = _pair(B, oracle, cfg, store_both=0)
    _cmp_solve(g, o, 1e-11, 1e-9, True)
    Q0, pa0, pb0 = g.density_operators()
    side = torch.cuda.Stream()
    with torch.cuda.stream(side):
        g2 = B.Fts(cfg.grid, cfg.cell, cfg.Ns, "diblock", **_kw(cfg))
        g2.set_fields(_dev(cfg.f0), _dev(cfg.f1))
        for _ in range(3):
            g2.propagate()
        Q1, pa1, pb1 = g2.density_operators()
    side.synchronize()
    assert Q1 == Q0 and torch.equal(pa1, pa0) and torch.equal(pb1, pb0)
    other = inputs.small_diblock(grid=(16, 16, 16), cell=(4.0, 4.0, 4.0), Ns=10, fA=0.4, seed=3)
    h, oh = _pair(B, oracle, other, store_both=0)
    for _ in range(3):                                 # alternate two contexts (each with its own graph)
        g.propagate(); h.propagate()
    oh.propagate()
    Qh, _, _ = h.density_operators(); Qo, _, _ = oh.density_operators()
    assert abs(Qh - Qo) < 1e-11 * abs(Qo) and g.density_operators()[0] == Q0
    for rep in range(25):
        t = B.Fts(cfg.grid, cfg.cell, cfg.Ns, "diblock", **_kw(cfg))
        t.set_fields(_dev(cfg.f0), _dev(cfg.f1))
        t.propagate(4); t.propagate()
        assert t.density_operators()[0] == Q0, rep
        t.close()


def test_state_is_invalidated_by_set_option_and_set_blocks(B, oracle):
    """After fts_cl_step, fts_operators reports the operators of the step's entry fields out of what the step left behind.  A
    change of plan (fts_set_option) or of the chain architecture (fts_set_blocks) invalidates that: FTS_ESTATE until the next
    solve, not numbers of the old chain.  Switching real_fields off ends the 'fields are not real' condition: the general path
    then works on the same complex fields without an fts_set_fields in between; a failed fts_set_option leaves the context usable."""
    cfg = inputs.small_diblock(grid=(16, 16, 16), Ns=12, fA=1.0 / 3.0)
    for change in (lambda g: g.set_option("lag", 1), lambda g: g.set_blocks([0, 1, 0], [2, 6, 4])):
        g, o = _pair(B, oracle, cfg)
        g.cl_step(0.01, 0, 5, 0)
        g.operators()                                   # allowed: the step's own solve
        g.cl_step(0.01, 0, 5, 1)
        change(g)
        with pytest.raises(B.FtsError) as e:
            g.operators()
        assert e.value.status == 2                      # FTS_ESTATE
        g.propagate()
        g.operators()
    g, o = _pair(B, oracle, cfg)                        # complex fields
    g.set_option("real_fields", 1)
    g.propagate()
    with pytest.raises(B.FtsError) as e:
        g.density_operators()
    assert e.value.status == 1                          # FTS_EINVAL: the declaration was wrong
    g.set_option("real_fields", 0)                      # ... and is withdrawn: no fts_set_fields needed
    _cmp_solve(g, o, 1e-11, 1e-9, True)
    with pytest.raises(B.FtsError) as e:
        g.set_option("march", 3)                        # TMA march on a 16^3 grid: refused, nothing changed
    assert e.value.status == 6
    g.propagate()
    Qg, _, _ = g.density_operators(); Qo, _, _ = o.density_operators()
    assert abs(Qg - Qo) <= 1e-11 * abs(Qo)
