"""PyTorch operator wrappers (paper_2412_10129_b200/autograd.py; section 2.8): the gradient autograd returns
for 1/2 ||A x - b||^2 is A^T (A x - b) as the oracle computes it with its exact transpose; second-order use (a gradient
through A^T) runs; the voxel-driven backprojector option gives the oracle's voxel-driven A^T."""
import numpy as np
import pytest

from oracle import oracle as orc
from tests import helpers as H
from workloads import make_config, phantom_for

pytestmark = pytest.mark.gpu

torch = pytest.importorskip("torch")


@pytest.fixture(scope="module")
def case():
    if not torch.cuda.is_available():
        pytest.skip("no CUDA device")
    geo, ang, rec = make_config("C1", scale=2, n_angles=12)
    vol = phantom_for(rec, geo).astype(np.float32)
    b = orc.ax(vol, geo, ang, orc.SIDDON)
    b = (b + 0.05 * b.max() * np.random.default_rng(0).standard_normal(b.shape)).astype(np.float32)
    return geo, ang, vol, b


@pytest.mark.parametrize("mode", ["siddon", "interp"])
def test_gradient_of_data_term_is_exact_transpose(case, mode):
    from paper_2412_10129_b200.autograd import Projector
    geo, ang, vol, b = case
    op = Projector(geo, ang, mode)
    x = torch.from_numpy(vol * 0.7).cuda().requires_grad_(True)
    loss = 0.5 * ((op(x) - torch.from_numpy(b).cuda()) ** 2).sum()
    loss.backward()
    om = orc.SIDDON if mode == "siddon" else orc.INTERP
    ref = orc.atb_exact(orc.ax(vol * 0.7, geo, ang, om) - b, geo, ang, om)
    assert H.rel_l2(x.grad.cpu().numpy().astype(np.float64), ref) <= (1e-5 if mode == "siddon" else 1e-4)


def test_backprojector_is_differentiable_and_matched_option(case):
    from paper_2412_10129_b200.autograd import Projector
    geo, ang, vol, b = case
    op = Projector(geo, ang, "siddon")
    y = torch.from_numpy(b).cuda().requires_grad_(True)
    w = torch.from_numpy(vol).cuda()
    (op.AT(y) * w).sum().backward()                                  # d/dy <A^T y, w> = A w
    assert H.rel_l2(y.grad.cpu().numpy().astype(np.float64), orc.ax(vol, geo, ang, orc.SIDDON)) <= 1e-5
    opm = Projector(geo, ang, "siddon", backprojector="matched")
    x = torch.from_numpy(vol).cuda().requires_grad_(True)
    (opm(x) * torch.from_numpy(b).cuda()).sum().backward()           # "gradient" with the voxel-driven pair: A^T_matched b
    assert H.rel_l2(x.grad.cpu().numpy().astype(np.float64), orc.atb(b, geo, ang, orc.MATCHED)) <= 1e-5
