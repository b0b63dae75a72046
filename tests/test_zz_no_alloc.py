"""shd_structure_factor_noalloc (include/shd.h): the allocation-free variant of shd_structure_factor, whose scratch is a
file-scope device array of libshd.so, against the existing path.  Collected last on purpose (the suite runs with
pytest -x); passes alone in a fresh process and after the other GPU tests."""
import numpy as np
import pytest

from paper_2304_09139_b200 import inputs

pytestmark = pytest.mark.gpu


@pytest.fixture(scope="module")
def shd():
    from paper_2304_09139_b200 import shd as m
    return m


def both_paths(shd, h, torch):
    S_ref, dev2_ref = h.structure_factor()                      # existing path: cudaMalloc'ed scratch, dev2 on the host
    S = torch.full((h.M,), float("nan"), dtype=torch.float64, device="cuda")
    dev2 = torch.full((2,), float("nan"), dtype=torch.float64, device="cuda")
    free0 = torch.cuda.mem_get_info()[0]
    h.structure_factor_noalloc(dev2, S)
    assert torch.cuda.mem_get_info()[0] == free0                # nothing was taken from (or returned to) the device
    # same kernels, same fixed reduction tree: the tolerance of the chunk / determinism tests, i.e. bit-identical
    assert torch.equal(S, S_ref)
    assert tuple(dev2.tolist()) == tuple(dev2_ref)
    return S_ref, dev2_ref


def test_no_alloc_structure_factor_matches_existing_path_twice(shd, oracle):
    import torch
    cfg = inputs.CONFIGS["cfg2"]
    h = shd.Shd(cfg.d, cfg.N, cfg.L, m_star=cfg.m_star)
    hi, lo = inputs.uniform_positions(cfg, 0)
    th, tl = shd.from_host(hi, lo)
    h.energy_grad(th, tl, want_grad=False)
    S1, d1 = both_paths(shd, h, torch)
    # second call in a row, on a SMALLER system after a different evaluation: the array still holds the first call's
    # block sums beyond this one's blocks, and none of them may leak into the result
    cfg1 = inputs.CONFIGS["cfg1"]
    h1 = shd.Shd(cfg1.d, cfg1.N, cfg1.L, m_star=cfg1.m_star)
    hi1, lo1 = inputs.uniform_positions(cfg1, 3)
    t1h, t1l = shd.from_host(hi1, lo1)
    h1.energy_grad(t1h, t1l, want_grad=False)
    S2, d2 = both_paths(shd, h1, torch)
    assert h1.M < h.M and d2 != d1
    # ... and against the oracle (Eq. 3), so that both paths being wrong together cannot pass
    n = oracle.enumerate_Q(cfg1.d, cfg1.m_star)
    re, im = oracle.rho(cfg1.d, cfg1.N, cfg1.L, hi1, lo1, n)
    So, dev2o = oracle.structure_factor(cfg1.N, re, im)
    assert np.abs(S2.cpu().numpy() - oracle.to_float(So)).max() <= 1e-14 * cfg1.N
    assert oracle.absdiff_dd(dev2o, [d2[0]], [d2[1]])[0] <= 1e-28 * cfg1.N ** 2 * len(n)
    # third call, back on the first handle, S not wanted, enqueue-only (wait = 0) then a stream synchronise
    dev2 = torch.zeros(2, dtype=torch.float64, device="cuda")
    h.structure_factor_noalloc(dev2, None, wait=False)
    torch.cuda.synchronize()
    assert tuple(dev2.tolist()) == tuple(d1)
    h.close()
    h1.close()


def test_no_alloc_rejects_what_it_cannot_hold(shd):
    import torch
    # a d = 2 wavevector table just beyond the limit (half space: n_0 = 1..1049, n_1 = -2000..1999); no evaluation is
    # needed, the size check comes first
    a, b = np.meshgrid(np.arange(1, 1050, dtype=np.int32), np.arange(-2000, 2000, dtype=np.int32), indexing="ij")
    big = shd.Shd(2, 8, 1.0, table=np.stack([a.ravel(), b.ravel()], axis=1))
    assert big.M == 1049 * 4000 > shd.SHD_NOALLOC_MAX_Q
    dev2 = torch.zeros(2, dtype=torch.float64, device="cuda")
    with pytest.raises(shd.ShdError) as e:
        big.structure_factor_noalloc(dev2)
    assert e.value.code == shd.SHD_EINVAL and "SHD_NOALLOC_MAX_Q" in str(e.value)
    big.close()
    h = shd.Shd(2, 16, 4.0, m_star=4)
    assert shd.lib.shd_structure_factor_noalloc(h._h, None, None, 1) == shd.SHD_EINVAL      # dev2 is required
    with pytest.raises(ValueError):
        h.structure_factor_noalloc(torch.zeros(2, dtype=torch.float64))                     # a host tensor is refused
    h.close()
