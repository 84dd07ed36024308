"""The seeded input generators (paper_1206_0675_b200.inputs): reproducibility, group properties and the
agreement of the numpy and torch back ends.  No method arithmetic is involved."""
import numpy as np
import pytest

from paper_1206_0675_b200 import inputs


def _unitarity(U):
    return float(np.abs(U @ np.conj(np.swapaxes(U, -1, -2)) - np.eye(3)).max())


def test_streams_are_counter_based():
    a = inputs.uniforms(11, inputs.STREAM_H, 0, 1000)
    b = np.concatenate([inputs.uniforms(11, inputs.STREAM_H, 0, 400), inputs.uniforms(11, inputs.STREAM_H, 400, 600)])
    assert np.array_equal(a, b) and 0.0 < a.min() and a.max() < 1.0
    assert not np.array_equal(a, inputs.uniforms(12, inputs.STREAM_H, 0, 1000))
    assert not np.array_equal(a, inputs.uniforms(11, inputs.STREAM_HAAR, 0, 1000))
    n = inputs.normals(3, 1, 0, 200000)
    assert abs(n.mean()) < 0.01 and abs(n.std() - 1.0) < 0.01


@pytest.mark.parametrize("name", ["C1"])
def test_named_configs_are_su3_and_reproducible(name):
    U = inputs.make_config(name)
    dims = inputs.CONFIGS[name]["dims"]
    assert U.shape == (dims[3], dims[2], dims[1], dims[0], 4, 3, 3)
    assert _unitarity(U) < 1e-13 and np.abs(np.linalg.det(U) - 1).max() < 1e-13
    assert np.array_equal(U, inputs.make_config(name))
    assert not np.array_equal(U, inputs.make_config(name, seed_offset=1))


def test_torch_backend_draws_the_same_streams():
    import torch

    a = inputs.uniforms(5, 3, 100, 4096)
    b = inputs._torch_uniforms(torch, 5, 3, 100, 4096, "cpu").numpy()
    assert np.array_equal(a, b)                       # the integer pipeline is bit-identical
    na = inputs.normals(5, 3, 7, 4096)
    nb = inputs._torch_normals(torch, 5, 3, 7, 4096, "cpu").numpy()
    assert np.max(np.abs(na - nb)) < 1e-13


def test_torch_hot_config_matches_numpy_hot_config():
    """Gram-Schmidt on the columns of the Ginibre matrix = its QR factor with positive diagonal (R21)."""
    dims = (4, 2, 6, 3)
    A = inputs.hot_config(dims, 1006)
    B = inputs.hot_config_torch(dims, 1006).numpy()
    assert A.shape == B.shape
    assert np.max(np.abs(A - B)) < 1e-13
    assert _unitarity(B) < 5e-15 and np.abs(np.linalg.det(B) - 1).max() < 5e-15
    # chunking changes at most the last bits (vectorised log / cos), never the stream positions
    C = inputs.hot_config_torch(dims, 1006, chunk=37).numpy()
    assert np.max(np.abs(B - C)) < 1e-14
