"""The seeded input generators produce what BASELINE.json:configs prescribe.  CPU only."""
import numpy as np
import pytest

import lattice_inputs as li


def dag(a):
    return np.conj(np.swapaxes(a, -1, -2))


@pytest.mark.parametrize("N", [2, 3, 4])
@pytest.mark.parametrize("kind", ["haar", "near"])
def test_links_are_special_unitary(N, kind):
    dims = (2, 2, 4, 4)
    U = li.haar_links(3, N, dims) if kind == "haar" else li.near_identity_links(3, N, dims, 0.3)
    assert U.shape == (64, 4, N, N)
    assert np.abs(U @ dag(U) - np.eye(N)).max() < 1e-13
    assert np.abs(np.linalg.det(U) - 1).max() < 1e-13
    if kind == "near":
        # exp(i eps H) with H Hermitian traceless: close to 1 but not 1, and -i log U / eps is Hermitian traceless
        dist = np.abs(U - np.eye(N)).max(axis=(-1, -2))
        assert 0.01 < dist.mean() < 1.0
        w, v = np.linalg.eig(U)
        H = (v * (np.angle(w) / 0.3)[..., None, :]) @ np.linalg.inv(v)
        assert np.abs(np.trace(H, axis1=-2, axis2=-1)).max() < 1e-10
        assert np.abs(H - dag(H)).max() < 1e-9


def test_counter_based_chunks_and_seeds():
    a = li.haar_matrices(9, 3, 100)
    b = np.concatenate([li._sun(9, li.STREAM_GAUGE, 0, 0.0, 3, 0, 37), li._sun(9, li.STREAM_GAUGE, 0, 0.0, 3, 37, 63)])
    assert np.array_equal(a, b)
    assert not np.array_equal(a, li.haar_matrices(10, 3, 100))
    s = li.gaussian_spinor(5, 50, 3)
    s2 = np.concatenate([li.gaussian_spinor(5, 20, 3), li.gaussian_spinor(5, 30, 3, first_site=20)])
    assert np.array_equal(s, s2)


def test_gaussian_moments():
    s = li.gaussian_spinor(77, 40000, 3).reshape(-1)
    for part in (s.real, s.imag):
        assert abs(part.mean()) < 0.01
        assert abs(part.var() - 1) < 0.01
        assert abs((part ** 4).mean() - 3) < 0.1
    assert abs(np.mean(s.real * s.imag)) < 0.01


def test_haar_moments():
    """Haar on SU(N): E U_ij = 0, E |U_ij|^2 = 1/N, E |tr U|^2 = 1."""
    for N in (2, 3):
        U = li.haar_matrices(78, N, 40000)
        assert np.abs(U.mean(axis=0)).max() < 0.01
        assert np.abs((np.abs(U) ** 2).mean(axis=0) - 1 / N).max() < 0.01
        tr = np.trace(U, axis1=-2, axis2=-1)
        assert abs((np.abs(tr) ** 2).mean() - 1) < 0.03
