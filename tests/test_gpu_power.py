"""GPU-vs-oracle parity of the power calculation: bit-exact."""
import numpy as np
import pytest

import oracle

pytestmark = pytest.mark.gpu


@pytest.mark.parametrize("n", [0, 1, 7, 4096, 1000003])
def test_power_bit_exact(n):
    import torch
    import paper_1307_5700_b200 as m
    g = np.random.default_rng(n)
    v = g.integers(-32768, 32768, size=(n, 2)).astype(np.int16)
    if n >= 7:
        v[:5] = [[-32768, -32768], [32767, 32767], [0, 0], [3, 4], [-32768, 32767]]      # extremes and the worked values
    dv = torch.from_numpy(v).cuda() if n else torch.zeros((4, 2), dtype=torch.int16, device="cuda")
    dp = torch.full((max(n, 4) + 8,), -7.0, dtype=torch.float32, device="cuda")
    m.mdsm_power_i16(dv, dp, n)
    torch.cuda.synchronize()
    got = dp.cpu().numpy()
    assert np.array_equal(got[:n], oracle.power_i16(v)) and np.all(got[n:] == -7.0)


def test_power_argument_errors():
    import torch
    import paper_1307_5700_b200 as m
    dv = torch.zeros((64, 2), dtype=torch.int16, device="cuda")
    dp = torch.zeros(64, dtype=torch.float32, device="cuda")
    with pytest.raises(m.MdsmError):
        m.mdsm_power_i16(dv, dp, -1)
    with pytest.raises(m.MdsmError):
        m.mdsm_power_i16(dv[1:], dp, 8)             # 4 bytes off a 16-byte boundary
