"""Pins for the CPU oracle (SURVEY.md sect. 8(c), P1-P9): the oracle is checked against things other
than itself -- numpy's FFT (library routine), hand-derived closed forms, the brute-force truncated
convolution (the definition), algebraic invariants of the Poisson bracket.  CPU only."""
import os

import numpy as np
import pytest

import oracle
from paper_1310_1485_b200 import workloads as W

GOLDEN = os.path.join(os.path.dirname(__file__), "golden")
LENGTHS = [24, 96, 144, 192, 384, 768]


def rel(a, b):
    return np.linalg.norm(a - b) / max(np.linalg.norm(b), 1e-300)


def planes_of(wl):
    chi, g, rhs = W.make_inputs(wl)
    G = W.as_planes(g, wl).numpy()
    X = W.as_planes(chi, wl).numpy()
    R = W.as_planes(rhs, wl).numpy()
    ci = np.array([W.chi_plane_of(wl, p) for p in range(wl.planes)])
    return X, G, R, ci


def bracket(X, G, wl, backend=oracle.DFT_RECURSIVE, scale=1.0):
    """N(X, G) per plane through the pseudo-spectral oracle with rhs = 0."""
    return oracle.nl_pseudospectral(X, G, np.zeros_like(G), scale, wl.kxmin, wl.kymin, backend=backend)


# ----------------------------------------------------------------------------- P9: 1-D DFT pins
@pytest.mark.parametrize("n", LENGTHS + [1, 2, 3, 5, 7, 12, 18])
def test_dft_matches_numpy_library(n):
    rng = np.random.default_rng(n)
    x = rng.standard_normal(n) + 1j * rng.standard_normal(n)
    for backend in (oracle.DFT_NAIVE, oracle.DFT_RECURSIVE):
        assert rel(oracle.dft(x, -1, backend), np.fft.fft(x)) < 1e-13
        assert rel(oracle.dft(x, +1, backend), np.fft.ifft(x) * n) < 1e-13


@pytest.mark.parametrize("n", LENGTHS)
def test_dft_recursive_vs_naive_and_closed_forms(n):
    rng = np.random.default_rng(100 + n)
    x = rng.standard_normal(n) + 1j * rng.standard_normal(n)
    for sign in (-1, +1):
        a = oracle.dft(x, sign, oracle.DFT_NAIVE)
        b = oracle.dft(x, sign, oracle.DFT_RECURSIVE)
        assert rel(b, a) < 1e-13
        # Parseval
        assert abs(np.vdot(b, b).real - n * np.vdot(x, x).real) < 1e-10 * n * np.vdot(x, x).real
        # round trip = N * identity
        assert rel(oracle.dft(b, -sign, oracle.DFT_RECURSIVE) / n, x) < 1e-13
    # delta at position s -> pure phase exp(sign*2*pi*i*s*k/n); delta at 0 -> constant 1
    for s in (0, 1, n // 3):
        d = np.zeros(n, complex)
        d[s] = 1.0
        k = np.arange(n)
        for sign in (-1, +1):
            want = np.exp(sign * 2j * np.pi * ((s * k) % n) / n)
            assert np.abs(oracle.dft(d, sign, oracle.DFT_RECURSIVE) - want).max() < 1e-14


# ------------------------------------------------------- P2: single-mode closed form (hand-derived)
def test_golden_single_mode_example():
    grid, ent = None, {"chi": [], "g": [], "N": []}
    for line in open(os.path.join(GOLDEN, "single_mode_example.txt")):
        t = line.split()
        if not t or t[0].startswith("#"):
            continue
        if t[0] == "grid":
            grid = (int(t[1]), int(t[2]), float(t[3]), float(t[4]))
        else:
            ent[t[0]].append((int(t[1]), int(t[2]), complex(float(t[3]), float(t[4]))))
    nx0, nky0, kxmin, kymin = grid
    X = np.zeros((nky0, nx0), complex)
    G = np.zeros((nky0, nx0), complex)
    for i, j, v in ent["chi"]:
        X[j, i] = v
    for i, j, v in ent["g"]:
        G[j, i] = v
    want = np.zeros((nky0, nx0), complex)
    for i, j, v in ent["N"]:
        want[j, i] = v
    for backend in (oracle.DFT_NAIVE, oracle.DFT_RECURSIVE):
        got = oracle.nl_pseudospectral(X, G, np.zeros_like(G), 1.0, kxmin, kymin, backend=backend)[0]
        assert np.abs(got - want).max() < 1e-15
    assert np.abs(oracle.nl_convolution_plane(X, G, kxmin, kymin) - want).max() < 1e-15


def closed_form_single_mode(nx0, nky0, kxmin, kymin, a1, b1, A, a2, b2, B):
    """Stored half-plane of N for chi = A e^{i k1.x} + c.c., g = B e^{i k2.x} + c.c. (b1, b2 > 0)."""
    amax, bmax = nx0 // 2 - 1, nky0 - 1
    C = (kymin * b1) * (kxmin * a2) - (kxmin * a1) * (kymin * b2)
    out = np.zeros((nky0, nx0), complex)

    def put(a, b, v):
        if abs(a) <= amax and 0 <= b <= bmax:
            out[b, a % nx0] += v

    put(a1 + a2, b1 + b2, C * A * B)
    if b1 - b2 > 0:
        put(a1 - a2, b1 - b2, -C * A * np.conj(B))
    elif b1 - b2 < 0:
        put(a2 - a1, b2 - b1, -C * np.conj(A) * B)
    else:  # ky = 0 column holds both signs of kx
        put(a1 - a2, 0, -C * A * np.conj(B))
        if a1 != a2:
            put(a2 - a1, 0, -C * np.conj(A) * B)
    return out


@pytest.mark.parametrize("nx0,nky0,kxmin,kymin", [(16, 8, 0.1, 0.1), (12, 6, 0.3, 0.07), (32, 16, 0.05, 0.2)])
def test_single_mode_closed_form_random_modes(nx0, nky0, kxmin, kymin):
    rng = np.random.default_rng(nx0 * 100 + nky0)
    amax, bmax = nx0 // 2 - 1, nky0 - 1
    cases = [(2, 3, 2, 3), (1, 2, -3, 2), (amax, bmax, amax, bmax), (-amax, 1, amax, bmax), (3, 1, 3, 1)]
    for _ in range(12):
        cases.append((rng.integers(-amax, amax + 1), rng.integers(1, bmax + 1),
                      rng.integers(-amax, amax + 1), rng.integers(1, bmax + 1)))
    for a1, b1, a2, b2 in cases:
        a1, b1, a2, b2 = int(a1), int(b1), int(a2), int(b2)
        A = complex(rng.standard_normal(), rng.standard_normal())
        B = complex(rng.standard_normal(), rng.standard_normal())
        X = np.zeros((nky0, nx0), complex)
        G = np.zeros((nky0, nx0), complex)
        X[b1, a1 % nx0] = A
        G[b2, a2 % nx0] = B
        want = closed_form_single_mode(nx0, nky0, kxmin, kymin, a1, b1, A, a2, b2, B)
        scale_ref = abs(A) * abs(B) * kxmin * kymin * amax * bmax
        got = oracle.nl_pseudospectral(X, G, np.zeros_like(G), 1.0, kxmin, kymin, backend=oracle.DFT_NAIVE)[0]
        assert np.abs(got - want).max() < 1e-13 * max(scale_ref, 1e-3), (a1, b1, a2, b2)
        got_c = oracle.nl_convolution_plane(X, G, kxmin, kymin)
        assert np.abs(got_c - want).max() < 1e-13 * max(scale_ref, 1e-3), (a1, b1, a2, b2)


# ------------------------------------------------ P1: pseudo-spectral route == the definition
def test_config0_all_planes_vs_convolution():
    wl = W.CONFIGS[0]
    X, G, R, ci = planes_of(wl)
    for backend in (oracle.DFT_NAIVE, oracle.DFT_RECURSIVE):
        out = oracle.nl_pseudospectral(X, G, R, wl.scale, wl.kxmin, wl.kymin, ci, backend)
        for p in range(wl.planes):
            N = oracle.nl_convolution_plane(X[ci[p]], G[p], wl.kxmin, wl.kymin)
            assert rel(out[p] - R[p], wl.scale * N) < 5e-14


@pytest.mark.parametrize("nx0,nky0,kxmin,kymin,chi_has_v", [
    (12, 6, 0.3, 0.07, False), (32, 16, 0.05, 0.2, True), (8, 4, 1.0, 1.0, False), (24, 2, 0.1, 0.5, True)])
def test_odd_shapes_vs_convolution(nx0, nky0, kxmin, kymin, chi_has_v):
    wl = W.small_workload(nx0, nky0, 2, 2, 1, 1, kxmin, kymin, chi_has_v, seed=nx0 + nky0)
    X, G, R, ci = planes_of(wl)
    out = oracle.nl_pseudospectral(X, G, R, wl.scale, wl.kxmin, wl.kymin, ci)
    for p in range(wl.planes):
        N = oracle.nl_convolution_plane(X[ci[p]], G[p], wl.kxmin, wl.kymin)
        assert rel(out[p] - R[p], wl.scale * N) < 5e-14
        # sampled-mode entry point agrees with the whole-plane one
        ii = np.array([0, 1, nx0 - 1, nx0 // 2, nx0 // 2 - 1])
        jj = np.array([0, nky0 - 1, 1, 0, nky0 // 2])
        assert np.array_equal(oracle.nl_convolution_modes(X[ci[p]], G[p], kxmin, kymin, ii, jj), N[jj, ii])


def numpy_fft_route(X, G, wl):
    """Independent re-statement with numpy's irfft2/rfft2 (library routine as a step)."""
    nx0, nky0, Nx, Ny = wl.nx0, wl.nky0, wl.Nx, wl.Ny
    kx, ky = W.kx_grid(wl).numpy(), W.ky_grid(wl).numpy()
    h = nx0 // 2

    def real(F, d):
        D = 1j * (kx[None, :] if d == 0 else ky[:, None]) * F
        S = np.zeros((Ny // 2 + 1, Nx), complex)
        S[:nky0, :h] = D[:, :h]
        S[:nky0, Nx - h + 1:] = D[:, h + 1:]
        return np.fft.irfft2(S.T, s=(Nx, Ny)) * Nx * Ny

    N = real(X, 0) * real(G, 1) - real(X, 1) * real(G, 0)
    Nh = np.fft.rfft2(N) / (Nx * Ny)
    out = np.zeros((nky0, nx0), complex)
    out[:, :h] = Nh[:h, :nky0].T
    out[:, h + 1:] = Nh[Nx - h + 1:, :nky0].T
    return out


@pytest.mark.parametrize("nx0,nky0", [(16, 8), (64, 32), (96, 48), (128, 32)])
def test_vs_numpy_library_route(nx0, nky0):
    wl = W.small_workload(nx0, nky0, 1, 2, 1, 1, 0.05, 0.04, True, seed=7)
    X, G, R, ci = planes_of(wl)
    out = oracle.nl_pseudospectral(X, G, R, wl.scale, wl.kxmin, wl.kymin, ci)
    for p in range(wl.planes):
        assert rel(out[p] - R[p], wl.scale * numpy_fft_route(X[p], G[p], wl)) < 1e-13


def test_sampled_modes_of_a_config1_plane_vs_convolution():
    """At configs[1] plane size the definition is affordable for a handful of output modes."""
    wl = W.small_workload(128, 32, 1, 1, 1, 1, 0.05, 0.05, True, seed=2)
    X, G, R, ci = planes_of(wl)
    out = oracle.nl_pseudospectral(X, G, R, wl.scale, wl.kxmin, wl.kymin, ci)
    ii = np.array([0, 1, 63, 65, 127, 17, 100, 40])
    jj = np.array([0, 31, 5, 0, 31, 16, 1, 30])
    N = oracle.nl_convolution_modes(X[0], G[0], wl.kxmin, wl.kymin, ii, jj)
    got = (out[0] - R[0])[jj, ii] / wl.scale
    assert np.abs(got - N).max() < 1e-12 * np.abs(N).max()


# ----------------------------------------------------------------- P3: antisymmetry
def test_antisymmetry_and_self_bracket():
    wl = W.small_workload(16, 8, 2, 2, 1, 1, 0.1, 0.13, True, seed=3)
    X, G, R, ci = planes_of(wl)
    Nxg = bracket(X, G, wl)
    Ngx = bracket(G, X, wl)
    assert np.abs(Nxg + Ngx).max() <= 1e-15 * np.abs(Nxg).max()
    assert np.abs(bracket(X, X, wl)).max() <= 1e-15 * np.abs(Nxg).max()
    for p in range(wl.planes):
        c1 = oracle.nl_convolution_plane(X[p], G[p], wl.kxmin, wl.kymin)
        c2 = oracle.nl_convolution_plane(G[p], X[p], wl.kxmin, wl.kymin)
        assert np.abs(c1 + c2).max() < 1e-14 * np.abs(c1).max()


# ------------------------------------------ P4/P5: Poisson-bracket invariants, N(0,0) = 0
def test_weighted_invariants_and_mean_mode():
    wl = W.CONFIGS[0]
    X, G, R, ci = planes_of(wl)
    N = bracket(X[ci], G, wl)
    w = np.full(wl.nky0, 2.0)
    w[0] = 1.0
    for p in range(wl.planes):
        for F in (X[ci[p]], G[p]):
            s = (w[:, None] * np.conj(F) * N[p]).sum()
            mag = (w[:, None] * np.abs(np.conj(F) * N[p])).sum()
            assert abs(s.real) < 1e-13 * mag
        assert abs(N[p][0, 0]) < 1e-14 * np.abs(N[p]).max()


# ------------------------------------- P6/P7: translation covariance, bilinearity, scale
def test_translation_covariance():
    wl = W.small_workload(16, 8, 1, 2, 1, 1, 0.1, 0.2, True, seed=5)
    X, G, R, ci = planes_of(wl)
    kx, ky = W.kx_grid(wl).numpy(), W.ky_grid(wl).numpy()
    phase = np.exp(1j * (kx[None, :] * 0.37 + ky[:, None] * (-1.21)))
    N0 = bracket(X, G, wl)
    N1 = bracket(X * phase, G * phase, wl)
    assert rel(N1, N0 * phase) < 1e-14


def test_bilinearity_and_scale():
    wl = W.small_workload(16, 8, 1, 2, 1, 1, 0.1, 0.2, True, seed=6)
    X, G, R, ci = planes_of(wl)
    N = bracket(X, G, wl)
    assert rel(bracket(2 * X, 3 * G, wl), 6 * N) < 1e-15
    X2, G2, _, _ = planes_of(W.small_workload(16, 8, 1, 2, 1, 1, 0.1, 0.2, True, seed=66))
    assert rel(bracket(X + X2, G, wl), N + bracket(X2, G, wl)) < 1e-14
    assert rel(bracket(X, G + G2, wl), N + bracket(X, G2, wl)) < 1e-14
    out = oracle.nl_pseudospectral(X, G, R, 0.7, wl.kxmin, wl.kymin)
    assert rel(out - R, 0.7 * N) < 1e-14
    assert np.array_equal(oracle.nl_pseudospectral(X, G, R, 0.0, wl.kxmin, wl.kymin), R)


# ------------------------------------------- P8 / R6 / R7: Hermitian column, Nyquist row
def test_output_ky0_hermitian_and_nyquist_untouched():
    wl = W.CONFIGS[0]
    X, G, R, ci = planes_of(wl)
    R = R.copy()
    R[:, :, wl.nx0 // 2] = 3.0 - 2.0j  # marker in the Nyquist row of rhs
    out = oracle.nl_pseudospectral(X, G, R, 1.0, wl.kxmin, wl.kymin, ci)
    assert np.array_equal(out[:, :, wl.nx0 // 2], R[:, :, wl.nx0 // 2])
    N = out - R
    h = wl.nx0 // 2
    col = N[:, 0, :]
    assert np.abs(col[:, h + 1:] - np.conj(col[:, 1:h][:, ::-1])).max() < 1e-14 * np.abs(N).max()
    assert np.abs(col[:, 0].imag).max() < 1e-14 * np.abs(N).max()


def test_nyquist_row_of_inputs_is_ignored():
    wl = W.small_workload(16, 8, 1, 2, 1, 1, 0.1, 0.1, True, seed=8)
    X, G, R, ci = planes_of(wl)
    base = oracle.nl_pseudospectral(X, G, R, 1.0, wl.kxmin, wl.kymin)
    Xn, Gn = X.copy(), G.copy()
    Xn[:, :, wl.nx0 // 2] = 5.0 + 1.0j
    Gn[:, :, wl.nx0 // 2] = -2.0 + 7.0j
    assert np.array_equal(oracle.nl_pseudospectral(Xn, Gn, R, 1.0, wl.kxmin, wl.kymin), base)
    for p in range(wl.planes):
        assert np.array_equal(oracle.nl_convolution_plane(Xn[p], Gn[p], wl.kxmin, wl.kymin),
                              oracle.nl_convolution_plane(X[p], G[p], wl.kxmin, wl.kymin))


def test_non_hermitian_ky0_column_real_part_reading():
    """R7: on a ky=0 column that is NOT Hermitian the real field is the real part of the synthesis;
    both routes implement that reading and agree."""
    wl = W.small_workload(16, 8, 1, 1, 1, 1, 0.1, 0.1, True, seed=9)
    X, G, R, ci = planes_of(wl)
    rng = np.random.default_rng(0)
    X = X.copy()
    G = G.copy()
    X[:, 0, :] = rng.standard_normal(16) + 1j * rng.standard_normal(16)
    G[:, 0, :] = rng.standard_normal(16) + 1j * rng.standard_normal(16)
    X[:, :, 8] = 0
    G[:, :, 8] = 0
    out = bracket(X, G, wl, backend=oracle.DFT_NAIVE)
    N = oracle.nl_convolution_plane(X[0], G[0], wl.kxmin, wl.kymin)
    assert rel(out[0], N) < 1e-13


def test_chi_broadcast_over_v_uses_the_right_chi_plane():
    wl = W.small_workload(16, 8, 3, 4, 2, 2, 0.1, 0.1, False, seed=10)
    X, G, R, ci = planes_of(wl)
    assert X.shape[0] == wl.nz * wl.nw * wl.nspec
    # p = z + nz*(v + nv*(w + nw*s))  ->  chi plane z + nz*(w + nw*s)
    for s in range(wl.nspec):
        for w in range(wl.nw):
            for v in range(wl.nv):
                for z in range(wl.nz):
                    p = z + wl.nz * (v + wl.nv * (w + wl.nw * s))
                    assert ci[p] == z + wl.nz * (w + wl.nw * s)
    out = oracle.nl_pseudospectral(X, G, R, wl.scale, wl.kxmin, wl.kymin, ci)
    p = 2 + wl.nz * (3 + wl.nv * (1 + wl.nw * 1))
    N = oracle.nl_convolution_plane(X[ci[p]], G[p], wl.kxmin, wl.kymin)
    assert rel(out[p] - R[p], wl.scale * N) < 5e-14
