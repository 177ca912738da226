"""GPU-vs-oracle parity of the mu-law quantiser (Eq. 5).  Both sides take the
quantisation decision in fp64; codes may differ only where 255 y / Xmax sits within 1e-9 of a half-integer."""
import numpy as np
import pytest

import oracle

pytestmark = pytest.mark.gpu


@pytest.mark.parametrize("n,mu", [(1, 255.0), (17, 255.0), (100003, 255.0), (1 << 20, 10.0), (4096, 1e-6)])
def test_mulaw_parity(n, mu):
    import torch
    import paper_1307_5700_b200 as m
    g = np.random.default_rng(n)
    x = (np.abs(g.normal(size=n)) * 30).astype(np.float32)
    if n > 16:
        x[3] = 0.0
        x[5] = -2.0
        x[7] = np.nan
    ref, xm = oracle.mulaw_u8(np.nan_to_num(x, nan=-1.0), mu)
    dx = torch.from_numpy(x).cuda()
    dc = torch.full((n + 16,), 77, dtype=torch.uint8, device="cuda")
    dm = torch.zeros(1, dtype=torch.float32, device="cuda")
    m.mdsm_mulaw_u8(dx, dc, n, mu, dm)
    torch.cuda.synchronize()
    got = dc.cpu().numpy()
    assert float(dm.item()) == xm == float(np.nanmax(x))
    v = 255.0 * np.log1p(mu * np.clip(np.nan_to_num(x, nan=0.0).astype(np.float64), 0, None) / xm) / np.log1p(mu)
    near = np.abs(v - np.floor(v) - 0.5) < 1e-9
    assert np.array_equal(got[:n][~near], ref[~near]) and np.all(np.abs(got[:n].astype(int) - ref.astype(int)) <= 1)
    assert np.all(got[n:] == 77)


def test_mulaw_all_zero_and_errors():
    import torch
    import paper_1307_5700_b200 as m
    dx = torch.zeros(64, dtype=torch.float32, device="cuda")
    dc = torch.full((64,), 9, dtype=torch.uint8, device="cuda")
    dm = torch.ones(1, dtype=torch.float32, device="cuda")
    m.mdsm_mulaw_u8(dx, dc, 64, 255.0, dm)
    torch.cuda.synchronize()
    assert float(dm.item()) == 0.0 and not dc.cpu().numpy().any()
    with pytest.raises(m.MdsmError):
        m.mdsm_mulaw_u8(dx, dc, 64, 0.0, dm)
    with pytest.raises(m.MdsmError):
        m.mdsm_mulaw_u8(dx, dc, -1, 255.0, dm)
