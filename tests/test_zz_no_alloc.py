"""GPU: dwf_norm2_static, the entry point that allocates nothing (its per-block partials live in a file-scope __device__
array of 32768 doubles, include/dwf.h), against the existing dwf_norm2 path -- same kernels, same summation order.

Collected last on purpose (the suite runs with pytest -x).  Passes alone in a fresh process (the address of the static array is
asked for on the first call) and after the other tests."""
import numpy as np
import pytest
import torch

from gpu_util import Rig

pytestmark = pytest.mark.gpu

from paper_2103_05034_b200 import DwfError  # noqa: E402
from paper_2103_05034_b200.dwf import DWF_EUNSUPPORTED  # noqa: E402

TOL = 1e-13          # the BLAS-1 reduction tolerance of tests/gpu_util.py (both sides accumulate in fp64)


@pytest.mark.parametrize("prec", ["f32", "f64"])
def test_norm2_static_matches_norm2_twice(prec):
    L, Ls, nrhs = (8, 8, 8, 8), 16, 3
    rig = Rig(L, Ls, prec, 0.01, seed_U=1001, ws_nrhs=nrhs)
    d = rig.d
    g = torch.Generator(device="cuda"); g.manual_seed(91)
    x1 = d.field(nrhs).normal_(generator=g)
    x2 = d.field(nrhs).normal_(generator=g) * 3.0            # other values: the shared scratch keeps the first call's partials
    out = torch.full((nrhs,), -1.0, dtype=torch.float64, device="cuda")
    for x in (x1, x2):                                        # two calls in a row
        want = np.array(d.norm2(x, nrhs))
        got = d.norm2_static(x, out, nrhs).cpu().numpy()      # .cpu() synchronises
        assert np.all(np.isfinite(got)) and np.all(got > 0)
        assert np.max(np.abs(got - want) / want) < TOL
        direct = (x.double() ** 2).sum().item()               # and both against a plain sum (all rhs together)
        assert abs(got.sum() - direct) / direct < 1e-12
    # half fields, one rhs: another launch geometry over the same array
    xh = d.field(1, half=True).normal_(generator=g)
    want = np.array(d.norm2(xh, 1, half=True))
    got = d.norm2_static(xh, out, 1, half=True).cpu().numpy()[:1]
    assert np.max(np.abs(got - want) / want) < TOL


def test_norm2_static_rejects_sizes_beyond_the_static_maximum():
    L, Ls, nrhs = (8, 8, 8, 8), 16, 32                        # 8 blocks per SM x 32 rhs x 2 doubles > 32768
    rig = Rig(L, Ls, "f32", 0.01, seed_U=1001)
    x = rig.d.field(nrhs).zero_()
    out = torch.zeros(nrhs, dtype=torch.float64, device="cuda")
    with pytest.raises(DwfError) as e:
        rig.d.norm2_static(x, out, nrhs)
    assert e.value.code == DWF_EUNSUPPORTED and "static maximum" in str(e.value)
    assert rig.d.norm2(x, nrhs) == [0.0] * nrhs               # the allocating path takes the same size
