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


def test_single_precision_database_is_the_fp64_database_rounded_once_to_nearest_even():
    """NEXT-1 (the stored values take about four bytes each): filter_store(single=True) must be the
    fp64 database -- pinned by the tests above -- rounded once per component to binary32, ties to even.  The rounding
    is re-derived here from the bit pattern of the double (integer arithmetic on the mantissa), not by calling the
    cast again; mode selection is untouched (same shape, zeros stay zeros)."""
    c, o = _setup()
    d64 = o.filter_store(*c["cut"])
    d32 = o.filter_store(*c["cut"], single=True)
    assert d32.dtype == np.complex64 and d32.shape == d64.shape

    def round_to_f32_bits(x):
        """IEEE round-to-nearest-even of positive normal doubles to binary32, from the bits."""
        b = np.abs(x).view(np.uint64)
        e = ((b >> np.uint64(52)) & np.uint64(0x7FF)).astype(np.int64) - 1023
        m = (b & np.uint64((1 << 52) - 1)) | np.uint64(1 << 52)                 # 53-bit significand
        keep, rest = m >> np.uint64(29), m & np.uint64((1 << 29) - 1)           # 24 bits kept, 29 dropped
        half = np.uint64(1 << 28)
        up = (rest > half) | ((rest == half) & ((keep & np.uint64(1)) == 1))
        keep = keep + up.astype(np.uint64)
        val = keep.astype(np.float64) * np.exp2((e - 23).astype(np.float64))     # exact: 25 bits times a power of two
        return np.sign(x) * val

    for part in (np.real, np.imag):
        x = part(d64).ravel()
        y = part(d32).ravel().astype(np.float64)
        normal = (np.abs(x) > 1e-30) & (np.abs(x) < 1e30)                      # binary32 normal range, far from its ends
        assert normal.sum() > 0.5 * x.size
        assert np.array_equal(y[normal], round_to_f32_bits(x[normal]))
        assert np.array_equal(y[x == 0.0], x[x == 0.0])
        assert np.abs(y[normal] - x[normal]).max() <= 2.0 ** -24 * np.abs(x[normal]).max()
    # ties go to even: 1 + 2^-24 -> 1, 1 + 3 * 2^-24 -> 1 + 2^-22 (hand values through the same helper and the cast)
    t = np.array([1.0 + 2.0 ** -24, 1.0 + 3.0 * 2.0 ** -24, 1.0 + 2.0 ** -24 + 2.0 ** -50])
    assert np.array_equal(round_to_f32_bits(t), np.array([1.0, 1.0 + 2.0 ** -22, 1.0 + 2.0 ** -23]))
    assert np.array_equal(t.astype(np.float32).astype(np.float64), round_to_f32_bits(t))


def test_run_emits_snapshots_at_the_cadence():
    """oracle.run == the plain loop of filter_store / stats_accumulate / step written out (L110-112)."""
    c, o = _setup()
    c2, ref = _setup()
    snaps = o.run(5, 2, 1, *c["cut"], single=True)
    want = []
    for n in range(5):
        ref.stats_accumulate()
        if n in (0, 2, 4):
            want.append(ref.filter_store(*c["cut"], single=True))
        ref.step()
    assert len(snaps) == 3 and all(np.array_equal(a, b) for a, b in zip(snaps, want))
    assert np.array_equal(o.stats_read()[0], ref.stats_read()[0]) and o.stats_read()[1] == 5
    assert np.array_equal(o.v, ref.v)
    assert o.run(2, 0, 0, *c["cut"]) == []


def test_spectra_sum_to_the_statistics_and_match_physical_space_transforms():
    """oracle.spectra (NEXT-4 "more statistics"): summed over their wavenumber the co-spectra are
    the plane statistics; and E_x of uu, vw equals the z-average of the one-dimensional x-transform of the PHYSICAL
    fields on the dealiased grid (an evaluation that never touches the spectral weights w_p), likewise E_z."""
    c, o = _setup()
    ex, ez = o.spectra()
    prof = o.stats_profiles()
    assert ex.shape == (7, o.ny, o.nx // 2) and ez.shape == (7, o.ny, o.nz)
    for n in range(7):
        sc = max(1.0, np.abs(prof[3 + n]).max())
        assert np.abs(ex[n].sum(axis=1) - prof[3 + n]).max() < 1e-12 * sc
        assert np.abs(ez[n].sum(axis=1) - prof[3 + n]).max() < 1e-12 * sc
    assert not ez[:, :, o.nz // 2].any()                                  # the z-Nyquist slot carries nothing
    u, v, w = (o.to_physical(f) for f in o.velocities_vorticities()[:3])     # [ny][mz][mx]
    mx, mz = o.mx, o.mz
    for n, (a, b) in ((0, (u, u)), (4, (v, w))):
        fa, fb = np.fft.fft(a, axis=2) / mx, np.fft.fft(b, axis=2) / mx     # full complex x-transform, all mx modes
        co = (fa * np.conj(fb)).real.mean(axis=1)                           # z-average -> [ny][mx]
        half = co[:, : o.nx // 2].copy()
        half[:, 1:] += co[:, :-(o.nx // 2):-1][:, : o.nx // 2 - 1]          # fold -p onto p
        assert np.abs(half - ex[n]).max() < 1e-12 * np.abs(ex[n]).max()
        ga, gb = np.fft.fft(a, axis=1) / mz, np.fft.fft(b, axis=1) / mz
        cz = (ga * np.conj(gb)).real.mean(axis=2)                           # x-average -> [ny][mz]
        slots = [q % mz for q in o.q]
        zz = cz[:, slots]
        zz[:, o.nz // 2] = 0.0
        # a real field's (-p, k_z) mode is the conjugate of (p, -k_z): the physical z-spectrum at k_z holds half of the
        # spectral weight-2 sums at k_z and half of those at -k_z, so compare the +-k_z pairs
        mirror = [list(o.q).index(-q) if s_ != o.nz // 2 else s_ for s_, q in enumerate(o.q)]
        assert np.abs((zz + zz[:, mirror]) - (ez[n] + ez[n][:, mirror])).max() < 1e-12 * np.abs(ez[n]).max()
