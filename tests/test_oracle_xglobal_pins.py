"""Pins for the x-global oracle (SURVEY.md sect. 8(f) f2; oracle/gene_nl_oracle.c, second half): checked against
numpy's FFT (library routine), a hand-derived closed form, the truncated convolution (the definition), Parseval's
identity for the ky = 0 output and the algebra of the product.  CPU only."""
import os

import numpy as np
import pytest

import oracle

GOLDEN = os.path.join(os.path.dirname(__file__), "golden")


def rnd(rng, nky0, nx, P=None):
    shape = (nky0, nx) if P is None else (P, nky0, nx)
    return rng.standard_normal(shape) + 1j * rng.standard_normal(shape)


def N_of(vex, vey, dxg, dyg, backend=oracle.DFT_RECURSIVE):
    nx = vex.shape[-1]
    return oracle.nlx_pseudospectral(vex, vey, dxg, dyg, np.ones(nx), np.zeros_like(vex), 1.0, backend=backend)


def rel(a, b):
    return np.linalg.norm(a - b) / max(np.linalg.norm(b), 1e-300)


@pytest.mark.parametrize("nky0,nx", [(4, 8), (8, 8), (16, 64), (5, 6), (32, 16), (48, 32)])
def test_algorithm_equals_definition(nky0, nx):
    rng = np.random.default_rng(100 * nky0 + nx)
    a, b, c, d = (rnd(rng, nky0, nx) for _ in range(4))
    ref = oracle.nlx_convolution_plane(a, b, c, d)
    for backend in (oracle.DFT_NAIVE, oracle.DFT_RECURSIVE):
        assert rel(N_of(a, b, c, d, backend), ref) < 5e-15


@pytest.mark.parametrize("nky0,nx", [(16, 64), (8, 4), (48, 8)])
def test_against_numpy_irfft_rfft(nky0, nx):
    """Independent restatement with a library routine: irfft over the zero-extended half spectrum."""
    rng = np.random.default_rng(7 + nky0)
    P = 3
    a, b, c, d = (rnd(rng, nky0, nx, P) for _ in range(4))
    pref = rng.standard_normal(nx)
    rhs = rnd(rng, nky0, nx, P)
    Ny = 3 * nky0

    def real(F):  # (P, nky0, nx) -> (P, Ny, nx), unnormalised synthesis
        return np.fft.irfft(F, n=Ny, axis=1) * Ny

    N = real(a) * real(c) + real(b) * real(d)
    ref = rhs + 0.7 * pref[None, None, :] * (np.fft.rfft(N, axis=1)[:, :nky0, :] / Ny)
    got = oracle.nlx_pseudospectral(a, b, c, d, pref, rhs, 0.7)
    assert rel(got, ref) < 1e-14


def test_worked_single_mode_example_from_golden_file():
    ent = {"vex": [], "vey": [], "dxg": [], "dyg": [], "N": []}
    for line in open(os.path.join(GOLDEN, "xglobal_single_mode_example.txt")):
        t = line.split()
        if not t or t[0].startswith("#"):
            continue
        if t[0] == "grid":
            nx, nky0 = int(t[1]), int(t[2])
        else:
            ent[t[0]].append((int(t[1]), int(t[2]), float(t[3]) + 1j * float(t[4])))
    f = {k: np.zeros((nky0, nx), complex) for k in ("vex", "vey", "dxg", "dyg")}
    for k in f:
        for x, j, v in ent[k]:
            f[k][j, x] = v
    expect = np.zeros((nky0, nx), complex)
    for x, j, v in ent["N"]:
        expect[j, x] = v
    for got in (N_of(f["vex"], f["vey"], f["dxg"], f["dyg"], oracle.DFT_NAIVE),
                oracle.nlx_convolution_plane(f["vex"], f["vey"], f["dxg"], f["dyg"])):
        assert np.abs(got - expect).max() < 1e-14


def test_random_single_modes_closed_form():
    rng = np.random.default_rng(3)
    nky0, nx = 16, 8
    for _ in range(40):
        k1, k2 = (int(v) for v in rng.integers(0, nky0, 2))
        x = int(rng.integers(0, nx))
        A, B = (complex(*rng.standard_normal(2)) for _ in range(2))
        a, c = np.zeros((nky0, nx), complex), np.zeros((nky0, nx), complex)
        a[k1, x], c[k2, x] = A, B
        z = np.zeros_like(a)
        expect = np.zeros_like(a)
        Ae = A.real if k1 == 0 else A        # Im of a ky = 0 entry is ignored
        Be = B.real if k2 == 0 else B
        w1 = 1 if k1 == 0 else 2             # number of exponentials of the real field
        w2 = 1 if k2 == 0 else 2
        # product of (Ae e^{ik1 y} [+ cc]) and (Be e^{ik2 y} [+ cc]), collected on stored modes j >= 0
        terms = [(k1 + k2, Ae * Be)]
        if w2 == 2:
            terms.append((k1 - k2, Ae * np.conj(Be)))
        if w1 == 2:
            terms.append((k2 - k1, np.conj(Ae) * Be))
        if w1 == 2 and w2 == 2:
            terms.append((-(k1 + k2), np.conj(Ae) * np.conj(Be)))
        for j, v in terms:
            if 0 <= j < nky0:
                expect[j, x] += v
        # each exponential pair lands once on j > 0 and, for j = 0, both members land there
        got = N_of(a, z, c, z, oracle.DFT_NAIVE)
        assert np.abs(got - expect).max() < 1e-13, (k1, k2)


def test_ky0_output_is_the_parseval_sum():
    """N^(x, 0) = <vex dxg + vey dyg>_y = Re sum_j w_j (vex_j conj(dxg_j) + ...), w_0 = 1 (real parts), w_j = 2."""
    rng = np.random.default_rng(11)
    nky0, nx = 16, 64
    a, b, c, d = (rnd(rng, nky0, nx) for _ in range(4))
    w = np.full(nky0, 2.0)
    w[0] = 0.0
    closed = (w[:, None] * (a * np.conj(c) + b * np.conj(d))).sum(0).real + a[0].real * c[0].real + b[0].real * d[0].real
    got = N_of(a, b, c, d)[0]
    assert np.abs(got.imag).max() < 1e-13 * np.abs(closed).max()
    assert np.abs(got.real - closed).max() < 1e-13 * np.abs(closed).max()


def test_algebra_of_the_product():
    rng = np.random.default_rng(5)
    nky0, nx = 16, 8
    a, b, c, d = (rnd(rng, nky0, nx) for _ in range(4))
    N = N_of(a, b, c, d)
    assert rel(N_of(c, d, a, b), N) < 1e-14                        # the product commutes
    assert rel(N_of(a, 0 * b, c, d) + N_of(0 * a, b, c, d), N) < 1e-14   # sum of the two terms
    assert rel(N_of(2 * a, 2 * b, 3 * c, 3 * d), 6 * N) < 1e-14    # bilinear
    a2 = a.copy()
    a2[0] += 1j * rng.standard_normal(nx)                          # Im of the ky = 0 row is ignored
    assert np.array_equal(N_of(a2, b, c, d), N)
    a3 = a.copy()
    a3[:, 5] = 0.0                                                 # x points do not talk to each other
    keep = np.arange(nx) != 5
    assert np.array_equal(N_of(a3, b, c, d)[:, keep], N[:, keep])


def test_prefactor_scale_and_accumulation():
    rng = np.random.default_rng(6)
    nky0, nx, P = 8, 16, 4
    a, b, c, d, rhs = (rnd(rng, nky0, nx, P) for _ in range(5))
    pref = rng.standard_normal(nx)
    N = oracle.nlx_pseudospectral(a, b, c, d, np.ones(nx), np.zeros_like(rhs), 1.0)
    out = oracle.nlx_pseudospectral(a, b, c, d, pref, rhs, -2.5)
    assert rel(out, rhs - 2.5 * pref[None, None, :] * N) < 1e-14
    assert np.array_equal(oracle.nlx_pseudospectral(a, b, c, d, pref, rhs, 0.0), rhs)   # scale = 0: bit-identical
    for p in range(P):                                             # planes are independent
        assert np.array_equal(oracle.nlx_pseudospectral(a[p], b[p], c[p], d[p], pref, rhs[p], -2.5), out[p])
