"""fts_mean_noalloc against the workspace path (collected last on purpose: `pytest -x` stops at the first failure, so a
failure in this add-on must not hide the parity tests; it passes alone in a fresh process and after the other files).

fts_mean_noalloc serves callers that have no device memory to lend the library and are not allowed to get any: an
observer inside another program's run that is handed slice pointers while all of HBM is already spoken for, or code that
cannot afford the device-wide synchronisation a cudaMalloc / cudaFree may cause while marches run on other streams
(include/fts.h).  Its reduction scratch is therefore one fixed array inside libfts.so, shared by every call on the device
and never cleared, so what has to be shown is (1) that it returns the Q the existing path computes in its workspace,
(2) that a call is not affected by what the call before it left in that array, and (3) that sizes beyond the stated
limit are refused.  Tolerances are the parity tests' own: 1e-11 relative on Q in complex128, 2e-4 in complex64.
"""
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


def _solved(B, grid, Ns, precision):
    """A diblock solve through the existing path: (Q it reports, its last slice q(x,1), the context)."""
    cfg = inputs.small_diblock(grid=grid, cell=(3.0, 4.0, 5.0), Ns=Ns, fA=0.4)
    dt = torch.complex128 if precision == "f64" else torch.complex64
    g = B.Fts(cfg.grid, cfg.cell, cfg.Ns, "diblock", precision=precision, fA=cfg.fA, chiN=cfg.chiN, B=cfg.B, Cc=cfg.C)
    dev = lambda a: torch.from_numpy(a).to("cuda:0").to(dt).contiguous()
    g.set_fields(dev(cfg.f0), dev(cfg.f1))
    g.propagate()
    Q, _, _ = g.density_operators()
    return Q, g.get_slice(0, Ns), g


def _as_complex(out):
    h = out.cpu()
    return complex(h[0].item(), h[1].item())


@pytest.mark.parametrize("precision", ["f64", "f32"])
def test_two_calls_in_a_row_match_the_workspace_path(B, precision):
    tol = 1e-11 if precision == "f64" else 2e-4
    # 64^3 fills all 592 partials of the static array, 16x8x8 then uses 4 of them: stale partials would show in the second mean
    Q_big, last_big, g_big = _solved(B, (64, 64, 64), 10, precision)
    Q_small, last_small, g_small = _solved(B, (16, 8, 8), 10, precision)
    out_big = torch.zeros(2, dtype=torch.float64, device="cuda:0")
    out_small = torch.zeros(2, dtype=torch.float64, device="cuda:0")
    B.mean_noalloc(last_big, out_big)            # first call in a fresh process: also the one-time address look-up
    torch.cuda.synchronize()
    free_before = torch.cuda.mem_get_info()[0]
    B.mean_noalloc(last_big, out_big)            # two calls back to back on one stream, no sync in between
    B.mean_noalloc(last_small, out_small)
    torch.cuda.synchronize()
    assert torch.cuda.mem_get_info()[0] >= free_before, "the entry point must not take device memory"
    m_big, m_small = _as_complex(out_big), _as_complex(out_small)
    assert abs(m_big - Q_big) <= tol * abs(Q_big), (m_big, Q_big)
    assert abs(m_small - Q_small) <= tol * abs(Q_small), (m_small, Q_small)
    # the same arithmetic as the workspace path, so in fact the same bits; and independent of it, the plain mean
    ref = last_small.to(torch.complex128).mean().item()
    assert abs(m_small - ref) <= 1e-13 * abs(ref)
    # and back to the long field: the short call must not have disturbed anything either
    again = torch.zeros(2, dtype=torch.float64, device="cuda:0")
    B.mean_noalloc(last_big, again)
    assert _as_complex(again) == m_big
    # the workspace path is untouched by all this: it still reports the same Q
    g_big.propagate()
    assert g_big.density_operators()[0] == Q_big
    del g_small


def test_sizes_beyond_the_limit_and_bad_arguments_are_refused(B):
    field = torch.ones(64, dtype=torch.complex128, device="cuda:0")
    out = torch.full((2,), -7.0, dtype=torch.float64, device="cuda:0")
    with pytest.raises(B.FtsError) as e:
        B.mean_noalloc(field, out, npoints=B.MEAN_NOALLOC_MAX_POINTS + 1)      # refused before anything is read
    assert e.value.status == 6 and "exceeds the limit" in str(e.value) and str(B.MEAN_NOALLOC_MAX_POINTS) in str(e.value)
    with pytest.raises(B.FtsError) as e:
        B.mean_noalloc(field, out, npoints=0)
    assert e.value.status == 1
    torch.cuda.synchronize()
    assert out.tolist() == [-7.0, -7.0]                                         # nothing was launched
    B.mean_noalloc(field, out)
    assert _as_complex(out) == 1.0 + 0.0j
    # exactly the limit (256^3 points, complex64) is accepted; the sums of these values are exact in fp64
    full = torch.full((B.MEAN_NOALLOC_MAX_POINTS,), 0.5 + 0.25j, dtype=torch.complex64, device="cuda:0")
    B.mean_noalloc(full, out)
    assert _as_complex(out) == 0.5 + 0.25j
