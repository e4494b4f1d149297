"""kf_mat66_multiply (layout micro-benchmark, sec. 4.3 Fig. 5) against the plain
definition, both layouts, ragged sizes.  fp32 products of six terms: |error| <= 6 * 2^-24 * sum |a||b| per element."""
import numpy as np
import pytest
import torch

from oracle import kf_oracle as o

pytestmark = pytest.mark.gpu


@pytest.mark.parametrize("n", [1, 31, 1000, 4099])
def test_mat66_both_layouts(n):
    from paper_1711_06571_b200 import binding as b
    rng = np.random.default_rng(n)
    A = rng.normal(size=(n, 6, 6)).astype(np.float32); B = rng.normal(size=(n, 6, 6)).astype(np.float32)
    ref = o.mat66_multiply(A, B)
    bound = 6 * 2.0 ** -24 * np.matmul(np.abs(A).astype(np.float64), np.abs(B).astype(np.float64)) + 1e-12
    # array of matrices
    c1 = b.kf_mat66_multiply(1, torch.from_numpy(A.reshape(n, 36)).cuda(), torch.from_numpy(B.reshape(n, 36)).cuda())
    # matrix-major, ld > n
    ld = (n + 31) // 32 * 32
    As = np.zeros((36, ld), np.float32); Bs = np.zeros((36, ld), np.float32)
    As[:, :n] = A.reshape(n, 36).T; Bs[:, :n] = B.reshape(n, 36).T
    c0 = torch.zeros((36, ld), dtype=torch.float32, device="cuda")
    dA, dB = torch.from_numpy(As).cuda(), torch.from_numpy(Bs).cuda()
    assert b.lib().kf_mat66_multiply(0, n, ld, dA.data_ptr(), dB.data_ptr(), c0.data_ptr(), None) == 0
    torch.cuda.synchronize()
    g1 = c1.cpu().numpy().reshape(n, 6, 6)
    g0 = c0.cpu().numpy()[:, :n].T.reshape(n, 6, 6)
    assert (np.abs(g1 - ref) <= bound).all() and (np.abs(g0 - ref) <= bound).all()
    assert np.array_equal(g0, g1)          # same arithmetic in both layouts


def test_mat66_arguments():
    from paper_1711_06571_b200 import binding as b
    x = torch.zeros((36, 32), dtype=torch.float32, device="cuda")
    assert b.lib().kf_mat66_multiply(0, 0, 0, None, None, None, None) == 0
    assert b.lib().kf_mat66_multiply(2, 4, 32, x.data_ptr(), x.data_ptr(), x.data_ptr(), None) == -1
    assert b.lib().kf_mat66_multiply(0, 64, 32, x.data_ptr(), x.data_ptr(), x.data_ptr(), None) == -1
    assert b.lib().kf_mat66_multiply(1, 4, 0, x.data_ptr() + 4, x.data_ptr(), x.data_ptr(), None) == -1
