"""The seeded input recipe (BASELINE.json configs[0]; readings R6/R9/R10)."""
import numpy as np
import torch

from paper_1310_1485_b200 import workloads as W


def test_config_table_matches_baseline_json():
    planes = [32, 8192, 8192, 24576, 73728]
    padded = [(24, 24), (192, 96), (384, 192), (768, 384), (144, 144)]
    for wl, P, (Nx, Ny) in zip(W.CONFIGS, planes, padded):
        assert wl.planes == P and (wl.Nx, wl.Ny) == (Nx, Ny)
    assert W.CONFIGS[1].chi_shape == (2, 8, 16, 32, 128)
    assert W.CONFIGS[1].plane_bytes * W.CONFIGS[1].planes == 512 * 2 ** 20
    assert W.CONFIGS[4].chi_has_v and W.CONFIGS[4].chi_shape == W.CONFIGS[4].g_shape


def test_recipe_properties_and_determinism():
    wl = W.CONFIGS[0]
    chi, g, rhs = W.make_inputs(wl)
    chi2, g2, rhs2 = W.make_inputs(wl)
    assert torch.equal(g, g2) and torch.equal(chi, chi2) and torch.equal(rhs, rhs2)
    assert g.shape == wl.g_shape and chi.shape == wl.chi_shape and g.dtype == torch.complex128
    assert torch.count_nonzero(rhs) == 0
    h = wl.nx0 // 2
    for t in (W.as_planes(g, wl), W.as_planes(chi, wl)):
        a = t.numpy()
        assert np.all(a[:, :, h] == 0)
        assert np.all(a[:, 0, 0].imag == 0)
        assert np.array_equal(a[:, 0, h + 1:], np.conj(a[:, 0, 1:h][:, ::-1]))
    kx = W.kx_grid(wl).numpy()
    assert np.allclose(kx[:8], 0.1 * np.arange(8)) and kx[8] == 0 and np.allclose(kx[9:], 0.1 * (np.arange(9, 16) - 16))
    # spectral fall-off: the high-k corner is damped relative to the low-k corner
    a = np.abs(W.as_planes(g, wl).numpy())
    assert a[:, 1, 1].mean() > 3 * a[:, 7, 7].mean()


def test_random_rhs_is_hermitian_consistent_without_falloff():
    wl = W.small_workload(16, 8, 2, 2, 2, 1, seed=4)
    chi, g, rhs = W.make_inputs(wl)
    r = W.as_planes(rhs, wl).numpy()
    h = wl.nx0 // 2
    assert np.all(r[:, :, h] == 0) and np.all(r[:, 0, 0].imag == 0)
    assert np.array_equal(r[:, 0, h + 1:], np.conj(r[:, 0, 1:h][:, ::-1]))
    assert 0.8 < r[:, 1:, :h].real.std() < 1.2
