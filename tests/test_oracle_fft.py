"""Pins for steps 2-4 of the oracle (padding, transforms, truncation) against brute-force DFT sums."""
import numpy as np

from oracle.channel import ChannelOracle
from paper_1808_06461_b200 import inputs


def _small(nx=8, ny=9, nz=4, lx=2 * np.pi, lz=np.pi):
    y = inputs.mesh_cosine(ny, 0.5)
    return ChannelOracle(nx, ny, nz, lx, lz, y, 100.0, 1e-3)


def _random_hermitian(o, rng):
    f = rng.standard_normal(o.v.shape) + 1j * rng.standard_normal(o.v.shape)
    nz = o.nz
    for q in range(1, nz // 2):
        f[nz - q, 0] = np.conj(f[q, 0])
    f[0, 0] = f[0, 0].real
    f[nz // 2] = 0
    return f


def test_to_physical_is_the_trigonometric_sum():
    """f(x_n,z_m) = sum_q [f(0,q) + 2 Re-part sum_{p>=1}] e^{i(kx x + kz z)} evaluated by brute force."""
    o = _small()
    rng = np.random.default_rng(3)
    f = _random_hermitian(o, rng)
    phys = o.to_physical(f)
    x = o.lx * np.arange(o.mx) / o.mx
    z = o.lz * np.arange(o.mz) / o.mz
    brute = np.zeros((o.ny, o.mz, o.mx))
    for s in range(o.nz):
        for p in range(o.nx // 2):
            e = np.exp(1j * (o.kx[p] * x[None, :] + o.kz[s] * z[:, None]))
            term = f[s, p, :, None, None] * e[None]
            brute += term.real if p == 0 else 2 * term.real
    assert np.abs(phys - brute).max() < 1e-12 * np.abs(brute).max()


def test_to_spectral_is_the_dft_sum_and_inverts():
    o = _small()
    rng = np.random.default_rng(4)
    r = rng.standard_normal((o.ny, o.mz, o.mx))
    s = o.to_spectral(r)
    x = o.lx * np.arange(o.mx) / o.mx
    z = o.lz * np.arange(o.mz) / o.mz
    for slot, p in ((0, 0), (1, 2), (3, 3), (3, 0), (2, 1)):
        e = np.exp(-1j * (o.kx[p] * x[None, :] + o.kz[slot] * z[:, None]))
        brute = (r * e[None]).sum(axis=(1, 2)) / (o.mx * o.mz)
        if slot == o.nz // 2:
            assert np.all(s[slot, p] == 0)
        else:
            assert np.abs(s[slot, p] - brute).max() < 1e-13
    f = _random_hermitian(o, rng)
    assert np.abs(o.to_spectral(o.to_physical(f)) - f).max() < 1e-13


def test_parseval_on_padded_grid():
    o = _small(nx=12, nz=8)
    rng = np.random.default_rng(5)
    a, b = _random_hermitian(o, rng), _random_hermitian(o, rng)
    pa, pb = o.to_physical(a), o.to_physical(b)
    wp = np.full(o.nx // 2, 2.0)
    wp[0] = 1.0
    spec = np.einsum("p,qpy->y", wp, (a * np.conj(b)).real)
    assert np.abs((pa * pb).mean(axis=(1, 2)) - spec).max() < 1e-12 * np.abs(spec).max()


def test_product_of_two_modes_is_dealiased():
    """PAPER.md L80 "fully dealiased by zero padding": the product of two retained modes lands on exactly the
    sum/difference modes with the analytic coefficients; out-of-range sums are dropped, never folded back."""
    o = _small(nx=8, nz=8)
    a = np.zeros(o.v.shape, complex)
    b = np.zeros(o.v.shape, complex)
    a[3, 3, :] = 1.0 + 2.0j   # (p,q) = (3,3): highest retained
    b[2, 2, :] = 0.5 - 1.0j   # (p,q) = (2,2)
    s = o.to_spectral(o.to_physical(a) * o.to_physical(b))
    # (a e^{i th1} + cc)(b e^{i th2} + cc) = ab e^{i(th1+th2)} + a b* e^{i(th1-th2)} + cc
    # sum mode (5,5) is outside the retained set (p<=3, |q|<=3) -> dropped; difference mode (1,1) kept.
    expect = np.zeros_like(s)
    expect[1, 1, :] = (1.0 + 2.0j) * np.conj(0.5 - 1.0j)
    assert np.abs(s - expect).max() < 1e-14
    # an aliasing transform (no padding) would fold (5,5) onto (p,q) = (3,-3)/(−3,3): check it is empty
    assert np.abs(s[o.nz - 3, 3]).max() < 1e-14
