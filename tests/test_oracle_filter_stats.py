"""Pins for the low-storage filter and the plane statistics."""
import numpy as np

from oracle.channel import ChannelOracle
from oracle import compact_fd as cfd
from paper_1808_06461_b200 import inputs


def _setup():
    c = inputs.config("cfg1")
    o = ChannelOracle(c["nx"], c["ny"], c["nz"], c["lx"], c["lz"], c["y"], c["re"], c["dt"])
    v, phi, omy = (t.numpy() for t in inputs.fluctuations(c))
    o.set_state(v * 50, phi * 50, omy * 50, c["U"], c["W"])  # O(5%) fluctuations so products matter
    return c, o


def test_second_order_consistency_of_the_database():
    """"Second-order consistent" (L124, L179): the (0,0) mode of every stored filtered product equals the
    full-field plane average, which equals the Parseval sum and the physical-grid mean."""
    c, o = _setup()
    out = o.filter_store(*c["cut"])
    prof = o.stats_profiles()
    assert out.shape == (10, o.ny, 2 * c["cut"][1] + 1, c["cut"][0] + 1)
    for n in range(10):
        assert np.abs(out[n, :, 0, 0].imag).max() < 1e-12 * max(1.0, np.abs(prof[n]).max())
        assert np.abs(out[n, :, 0, 0].real - prof[n]).max() < 1e-12 * max(1.0, np.abs(prof[n]).max()), n
    u, v, w, ox, oy, oz = (o.to_physical(f) for f in o.velocities_vorticities())
    phys = [u, v, w, u * u, u * v, u * w, v * v, v * w, w * w, ox * ox + oy * oy + oz * oz]
    for n in range(10):
        m = phys[n].mean(axis=(1, 2))
        assert np.abs(m - prof[n]).max() < 1e-12 * max(1.0, np.abs(m).max()), n
    assert np.abs(prof[0] - o.U).max() == 0.0 and np.abs(prof[1]).max() == 0.0


def test_filter_mode_selection_is_the_integer_predicate():
    """Reading R11: rectangular in index space, 0<=p<=Kx, |q|<=Kz, all y; stored u_i are plain copies."""
    c, o = _setup()
    kxc, kzc = 5, 3
    out = o.filter_store(kxc, kzc)
    u, v, w, *_ = o.velocities_vorticities()
    qs = list(range(0, kzc + 1)) + list(range(-kzc, 0))
    for n, f in enumerate((u, v, w)):
        for r, q in enumerate(qs):
            for p in range(kxc + 1):
                assert np.array_equal(out[n, :, r, p], f[q % o.nz, p, :])
    # a wider cutoff contains the narrower one bit for bit (sharp cutoff = pure selection)
    wide = o.filter_store(kxc + 2, kzc + 1)
    qs_w = list(range(0, kzc + 2)) + list(range(-kzc - 1, 0))
    for r, q in enumerate(qs):
        assert np.array_equal(wide[:, :, qs_w.index(q), : kxc + 1], out[:, :, r, :])


def test_filter_commutes_with_derivatives():
    """L124: the sharp cutoff "commutes with all the derivatives": filter(D f) == D filter(f) exactly."""
    c, o = _setup()
    kxc, kzc = 6, 4
    u = o.velocities_vorticities()[0]
    qs = [q % o.nz for q in list(range(0, kzc + 1)) + list(range(-kzc, 0))]

    def filt(f):
        return f[qs][:, : kxc + 1, :]

    assert np.array_equal(filt(o.D1(u)), cfd.d1(o.A1, o.B1, filt(u)))
    ikx = 1j * o.kx[None, :, None]
    ikz = 1j * o.kz[:, None, None]
    assert np.array_equal(filt(ikx * u), ikx[:, : kxc + 1] * filt(u))
    assert np.array_equal(filt(ikz * u), ikz[qs] * filt(u))


def test_stats_accumulate_read_reset():
    c, o = _setup()
    o.stats_accumulate()
    p1 = o.stats_profiles()
    o.substep()
    o.stats_accumulate()
    s, n = o.stats_read()
    assert n == 2 and np.allclose(s, p1 + o.stats_profiles(), rtol=0, atol=0)
    assert np.all(s[3] >= 0) and np.all(s[6] >= 0) and np.all(s[8] >= 0) and np.all(s[9] >= 0)
    o.stats_reset()
    assert o.stats_read()[1] == 0 and not o.stats_read()[0].any()
