"""GPU parity: the CUDA path (through the C ABI) against the CPU oracle on the same seeded inputs.

Tolerances (BASELINE.json north_star): relative L2 error 1e-11 per substep, 1e-8 after 10 full steps;
filter mode selection bit-exact.  Stage tests feed the library's stage hooks and the oracle the SAME
seeded synthetic arrays; nothing the oracle consumes comes from the CUDA path.
"""
import numpy as np
import pytest
import torch

import __graft_entry__ as entry
from oracle.channel import ChannelOracle
from paper_1808_06461_b200 import inputs

pytestmark = pytest.mark.gpu

TOL_SUBSTEP = 1e-11
TOL_10STEPS = 1e-8


@pytest.fixture(scope="module")
def B():
    if not torch.cuda.is_available():
        pytest.skip("no CUDA device")
    entry.build()
    from paper_1808_06461_b200 import binding
    return binding


def rel(a, b):
    a = a.cpu().numpy() if isinstance(a, torch.Tensor) else np.asarray(a)
    return float(np.linalg.norm((a - b).ravel()) / max(np.linalg.norm(np.asarray(b).ravel()), 1e-300))


def make(B, name, **over):
    c = inputs.config(name, **over)
    ch = B.Channel(c["nx"], c["ny"], c["nz"], c["lx"], c["lz"], c["y"], c["re"], c["dt"]).bind("cuda:0")
    o = ChannelOracle(c["nx"], c["ny"], c["nz"], c["lx"], c["lz"], c["y"], c["re"], c["dt"])
    return c, ch, o


def seeded_state(c, boost=1.0):
    v, phi, omy = (t.numpy() * boost for t in inputs.fluctuations(c))
    return v, phi, omy


# ---- fp64 rounding yardstick ------------------------------------------------------------------------------
# phi^ = lap(v^) comes out of Helmholtz problems whose condition number grows like 1/dy_min^2 and of the 2x2
# influence matrix, so BOTH fp64 evaluations (oracle and kernels) carry a rounding error on phi^ that can exceed
# north_star's 1e-11 per substep (on config 1 the oracle itself is 4e-11 away from the exact discrete solution after
# three substeps).  oracle.channel_hp.ChannelHP evaluates the same discrete steps in 80-bit long double (pinned
# against exact rational arithmetic in tests/test_oracle_hp.py); |oracle - hp| is the oracle's own rounding error on
# the given data.  Gate: |gpu - oracle| and |gpu - hp| <= max(1e-11 n, K_FLOOR |oracle - hp|).
K_FLOOR = 4.0
# the same per (kx,kz) line, so that low-energy modes are checked and not hidden in the whole-field norm
K_LINE = 16.0
ABS_LINE = 1e-11


def make_hp(o):
    from oracle.channel_hp import ChannelHP
    return ChannelHP(o)


def noise_floor(o, h):
    return {k: rel(getattr(o, k), np.asarray(getattr(h, k)).astype(np.asarray(getattr(o, k)).dtype)) for k in ("v", "phi", "omy", "U")}


def line_rel(a, b):
    """Relative L2 error of every (z slot, p) line: [nz][nxh]; lines where the reference vanishes count as 0."""
    a = a.cpu().numpy() if isinstance(a, torch.Tensor) else np.asarray(a)
    den = np.linalg.norm(b, axis=-1)
    return np.linalg.norm(a - b, axis=-1) / np.where(den > 0, den, 1.0)


def check_lines(gpu, o, h, nsub, where):
    """Per-line gate, so that low-energy modes are checked and not hidden in the whole-field norm: every line's relative
    error |gpu - oracle| <= max(1e-11 n, K_LINE x max(that line's |oracle - hp|, the median over lines of |oracle - hp|)).
    Lines on which the oracle itself is rounding noise (|oracle - hp| > 10% of the line: modes far below the eps U^2
    that the mean-flow products leak into every mode, a third of config 1's e^-70 spectrum) are skipped -- there is
    nothing to compare there; they stay covered by the whole-field norm.  Measured on config 1 and "mid"
    (profiles/r2_parity.md): |gpu - oracle| / |oracle - hp| per line has median 1.1, 99% quantile 5, maximum 9 on the
    compared lines; a mode-local defect (a wrong wavenumber, a dropped boundary row) is orders of magnitude above."""
    worst = {}
    for k, g in zip(("v", "phi", "omy"), gpu):
        ref = getattr(o, k)
        e = line_rel(g, ref)
        f = line_rel(np.asarray(getattr(h, k)).astype(complex), ref)
        live = (np.linalg.norm(ref, axis=-1) > 0) & (f <= 0.1)
        if not live.any():
            continue
        bound = np.maximum(TOL_SUBSTEP * nsub, K_LINE * np.maximum(f, np.median(f[live])))
        # weak lines: transform roundoff leaks eps x (strongest modes) into every mode (the oracle's own absolute error
        # on config 1's weak lines is up to 8e-12 of the strongest line, the kernels' -- twiddles by products, a few
        # ulp -- about twice that on some): an ABSOLUTE error below ABS_LINE = 1e-11 x the strongest line is within
        # north_star's tolerance whatever it is relative to a line 1e-8 times weaker
        nrm = np.linalg.norm(ref, axis=-1)
        bound = np.maximum(bound, ABS_LINE * nrm.max() / np.where(nrm > 0, nrm, 1.0))
        ratio = np.where(live, e / bound, 0.0)
        worst[k] = float(ratio.max())
        idx = np.unravel_index(np.argmax(ratio), ratio.shape)
        q = np.quantile((e / np.maximum(f, 1e-300))[live], [0.5, 0.99, 1.0])
        print(f"  lines {where} {k}: {int(live.sum())} compared, {int((~live).sum())} skipped; |gpu-oracle|/|oracle-hp| per line: "
              f"median {q[0]:.2f}, 99% {q[1]:.2f}, max {q[2]:.2f}; worst bound ratio {worst[k]:.2f}")
        assert worst[k] <= 1.0, (where, k, idx, float(e[idx]), float(f[idx]))
    return worst


def check_state(ch, o, h, nsub, where, lines=True):
    """Gate: relative L2 <= 1e-11 per substep (north_star), or, where the oracle's own fp64 rounding error on this
    data (|oracle - long-double evaluation|) is above that, <= K_FLOOR x that error; v and U are asserted against
    the plain tolerance by the callers."""
    gpu = ch.get_state()
    e = state_errors(ch, o, gpu)
    f = noise_floor(o, h) if h is not None else {k: 0.0 for k in ("v", "phi", "omy", "U")}
    for k, g in zip(("v", "phi", "omy", "U"), gpu):
        lim = max(TOL_SUBSTEP * nsub, K_FLOOR * f[k])
        assert e[k] < lim, (where, k, e, f)
        if h is not None:
            assert rel(g, np.asarray(getattr(h, k)).astype(np.asarray(getattr(o, k)).dtype)) < lim, (where, k, "vs hp", e, f)
    assert e["W"] < 1e-12, (where, e)
    if lines and h is not None:
        e["worst_line_ratio"] = check_lines(gpu[:3], o, h, nsub, where)
    print(f"{where}: |gpu-oracle| {e}  |oracle-hp| {f}")
    return e, f


def state_errors(ch, o, gpu=None):
    gv, gphi, gomy, gU, gW = gpu if gpu is not None else ch.get_state()
    return {"v": rel(gv, o.v), "phi": rel(gphi, o.phi), "omy": rel(gomy, o.omy), "U": rel(gU, o.U),
            "W": float(np.abs(gW.cpu().numpy() - o.W).max())}


@pytest.mark.parametrize("name", ["cfg1", "mid"])
def test_transposes_are_bit_exact(B, name):
    """a2/a8: line <-> plane layout is a pure permutation."""
    c, ch, o = make(B, name)
    g = torch.Generator().manual_seed(5)
    a = torch.view_as_complex(torch.randn(ch.shape + (2,), generator=g, dtype=torch.float64)).cuda()
    nm = ch.shape[0] * ch.shape[1]
    plane = torch.empty((c["ny"], nm), dtype=torch.complex128, device="cuda")
    back = torch.empty_like(a)
    ch.debug_transpose(0, a, plane)
    ch.debug_transpose(1, plane, back)
    torch.cuda.synchronize()
    assert torch.equal(plane, a.reshape(nm, c["ny"]).t().contiguous())
    assert torch.equal(back, a)
    ch.close()


@pytest.mark.parametrize("name,boost", [("cfg1", 50.0), ("mid", 1.0)])
def test_stage_derive(B, name, boost):
    """a1-a2: u, w, om_x, om_z from the state (readings R1, R7)."""
    c, ch, o = make(B, name)
    v, phi, omy = seeded_state(c, boost)
    ch.set_state(v, phi, omy, c["U"], c["W"])
    o.set_state(v, phi, omy, c["U"], c["W"])
    u, vv, w, ox, oy, oz = o.velocities_vorticities()
    for fid, ref in ((B.F_U, u), (B.F_W, w), (B.F_OMX, ox), (B.F_OMZ, oz), (B.F_V, vv), (B.F_OMY, oy)):
        assert rel(ch.debug_get_field(fid), ref) < 1e-13, fid
    ch.close()


@pytest.mark.parametrize("name", ["cfg1", "mid"])
def test_stage_nonlinear(B, name):
    """a3-a8: padded inverse FFTs, u x omega on the 3/2 grid, forward FFTs, truncation.  Inputs are six
    independent seeded random Hermitian fields (not a flow), so every mode and the padding are exercised."""
    c, ch, o = make(B, name)
    rng = np.random.default_rng(21)
    nz = c["nz"]
    fields = []
    for _ in range(6):
        f = rng.standard_normal(ch.shape) + 1j * rng.standard_normal(ch.shape)
        for q in range(1, nz // 2):
            f[nz - q, 0] = np.conj(f[q, 0])
        f[0, 0] = f[0, 0].real
        f[nz // 2] = 0
        fields.append(f)
    for fid, f in zip((B.F_U, B.F_V, B.F_W, B.F_OMX, B.F_OMY, B.F_OMZ), fields):
        ch.debug_set_field(fid, f)
    ch.debug_run_stage(B.STAGE_NONLINEAR)
    H = o.nonlinear(fields)
    for fid, ref in zip((B.F_H1, B.F_H2, B.F_H3), H):
        got = ch.debug_get_field(fid)
        assert rel(got, ref) < 1e-13, fid
        assert not got[nz // 2].any()      # z-Nyquist slot stays empty
    ch.close()


@pytest.mark.parametrize("name", ["cfg1", "mid"])
@pytest.mark.parametrize("isub", [0, 1, 2])
def test_stage_ysolve(B, name, isub):
    """a9-a12 for each of the three substep coefficient sets, from seeded H, state and history."""
    c, ch, o = make(B, name)
    v, phi, omy = seeded_state(c, 10.0)
    rng = np.random.default_rng(100 + isub)

    def rnd():
        f = rng.standard_normal(ch.shape) + 1j * rng.standard_normal(ch.shape)
        f[c["nz"] // 2] = 0
        return f

    H = [rnd() * 1e2 for _ in range(3)]
    for Hc in H:
        Hc[0, 0] = Hc[0, 0].real
    hvp, hgp = rnd(), rnd()
    hvp[0, 0] = hgp[0, 0] = 0
    ch.set_state(v, phi, omy, c["U"], c["W"])
    o.set_state(v, phi, omy, c["U"], c["W"])
    for fid, f in ((B.F_H1, H[0]), (B.F_H2, H[1]), (B.F_H3, H[2]), (B.F_HV_PREV, hvp), (B.F_HG_PREV, hgp)):
        ch.debug_set_field(fid, f)
    ch.debug_set_substep_index(isub)
    ch.debug_run_stage(B.STAGE_YSOLVE)
    # oracle: same substep with the nonlinear term replaced by the seeded H
    o.isub = isub
    o.hv_prev, o.hg_prev = hvp.copy(), hgp.copy()
    o.nonlinear = lambda fields: tuple(h.copy() for h in H)
    o.substep()
    e = state_errors(ch, o)
    assert max(e["v"], e["phi"], e["omy"], e["U"]) < TOL_SUBSTEP, e
    assert rel(ch.debug_get_field(B.F_HV_PREV), o.hv_prev) < 1e-12
    assert rel(ch.debug_get_field(B.F_HG_PREV), o.hg_prev) < 1e-13
    ch.close()


def test_config1_ten_substeps_filter_and_stats(B):
    """BASELINE config 1: 10 RK substeps at dt=1e-3, then the filter |kx|,|kz| <= 8 and the statistics."""
    c, ch, o = make(B, "cfg1")
    v, phi, omy = seeded_state(c)
    ch.set_state(v, phi, omy, c["U"], c["W"])
    o.set_state(v, phi, omy, c["U"], c["W"])
    t = make_hp(o)
    t.set_state(v, phi, omy, c["U"], c["W"])
    for n in range(10):
        ch.substep()
        o.substep()
        t.substep()
        e, f = check_state(ch, o, t, n + 1, n)
        # the primitive unknowns meet the stated tolerance outright
        assert max(e["v"], e["U"]) < TOL_SUBSTEP * (n + 1), (n, e)
    kxc, kzc = c["cut"]
    got = ch.filter_store(kxc, kzc).cpu().numpy()
    ref = o.filter_store(kxc, kzc)
    # mode selection: the stored velocities are bit-exact copies of the GPU's own retained modes ...
    u = ch.debug_get_field(B.F_U).cpu().numpy()
    qs = [q % c["nz"] for q in list(range(0, kzc + 1)) + list(range(-kzc, 0))]
    assert np.array_equal(got[0], np.transpose(u[qs][:, : kxc + 1, :], (2, 0, 1)))
    # ... and all ten variables agree with the oracle
    for n in range(10):
        assert rel(got[n], ref[n]) < 1e-10, n
    ch.stats(B.STATS_RESET)
    ch.stats(B.STATS_ACCUMULATE)
    prof, ns = ch.stats(B.STATS_READ)
    assert ns == 1
    pref = o.stats_profiles()
    for n in range(10):
        assert np.abs(prof[n] - pref[n]).max() < 1e-10 * max(1.0, np.abs(pref[n]).max()), n
    # second-order consistency on the GPU side: (0,0) mode of the stored products == plane statistics
    for n in range(3, 10):
        assert np.abs(got[n, :, 0, 0].real - prof[n]).max() < 1e-11 * max(1.0, np.abs(prof[n]).max())
    sc = ch.scalars()
    assert sc[0] == pytest.approx(o.pgrad, rel=1e-9) and sc[1] == pytest.approx(o.Q0, rel=1e-14)
    ch.close()


def test_mid_full_steps_filter_stats(B):
    """Mid-size case (96x65x48: several z tiles, ragged x tail, radix 2/3/4 mixes): 2 full steps."""
    c, ch, o = make(B, "mid")
    v, phi, omy = seeded_state(c)
    ch.set_state(v, phi, omy, c["U"], c["W"])
    o.set_state(v, phi, omy, c["U"], c["W"])
    t = make_hp(o)
    t.set_state(v, phi, omy, c["U"], c["W"])
    for n in range(2):
        ch.step()
        o.step()
        t.step()
        check_state(ch, o, t, 3 * (n + 1), n)
    got = ch.filter_store(*c["cut"]).cpu().numpy()
    ref = o.filter_store(*c["cut"])
    for n in range(10):
        assert rel(got[n], ref[n]) < 1e-10, n
    ch.stats(B.STATS_RESET | B.STATS_ACCUMULATE)
    ch.stats(B.STATS_ACCUMULATE)
    prof, ns = ch.stats(B.STATS_READ)
    assert ns == 2
    assert np.abs(prof / 2 - o.stats_profiles()).max() < 1e-10 * np.abs(prof).max()
    ch.close()


def test_ten_full_steps(B):
    """north_star: 1e-8 relative L2 after 10 full steps (config 1, fluctuations boosted to 5% so the
    nonlinear term matters)."""
    c, ch, o = make(B, "cfg1")
    v, phi, omy = seeded_state(c, 50.0)
    ch.set_state(v, phi, omy, c["U"], c["W"])
    o.set_state(v, phi, omy, c["U"], c["W"])
    h = make_hp(o)
    h.set_state(v, phi, omy, c["U"], c["W"])
    for _ in range(10):
        ch.step()
        o.step()
        h.step()
    e = state_errors(ch, o)
    assert max(e["v"], e["phi"], e["omy"], e["U"]) < TOL_10STEPS, e
    # per line as well (low-energy modes), against the oracle's own accumulated rounding error on each line
    w = check_lines(ch.get_state()[:3], o, h, 30, "ten steps")
    print("ten full steps: |gpu-oracle|", e, " |oracle-hp|", noise_floor(o, h), " worst line ratio", w)
    ch.close()


def test_poiseuille_steady_on_gpu(B):
    c, ch, o = make(B, "cfg1")
    z = np.zeros(ch.shape, complex)
    ch.set_state(z, z, z, c["U"], c["W"])
    for _ in range(5):
        ch.step()
    gv, gphi, gomy, gU, gW = ch.get_state()
    assert float(gv.abs().max()) == 0.0 and float(gomy.abs().max()) == 0.0
    assert np.abs(gU.cpu().numpy() - c["U"]).max() < 1e-10
    assert ch.scalars()[0] == pytest.approx(2.0 * 90.0 / 180.0, rel=1e-7)
    ch.close()


def test_orr_sommerfeld_growth_on_gpu(B):
    """BASELINE config 2 in full: 667 steps (2001 substeps, reading R15) of the alpha=1 mode at Re=7500."""
    import os
    from oracle.os_mode import discrete_os_mode
    c, ch, o = make(B, "cfg2")
    gold = [l for l in open(os.path.join(os.path.dirname(__file__), "golden", "os_re7500_alpha1.txt")) if l[0] != "#"][0].split()
    gold = float(gold[0]) + 1j * float(gold[1])
    sig, v, phi = discrete_os_mode(o.y, o.A1, o.B1, o.A2, o.B2, c["U"], o.kx[1], o.nu, gold)
    V = np.zeros(ch.shape, complex)
    P = np.zeros(ch.shape, complex)
    V[0, 1], P[0, 1] = 1e-6 * v, 1e-6 * phi
    ch.set_state(V, P, 0 * V, c["U"], c["W"])
    nst = 667
    for _ in range(nst):
        ch.step()
    gv = ch.get_state()[0].cpu().numpy()
    r = np.vdot(V[0, 1], gv[0, 1]) / np.vdot(V[0, 1], V[0, 1])
    sig_num = np.log(r) / (nst * c["dt"])
    # log of a complex ratio: the phase wraps; compare growth directly and frequency modulo 2 pi / T
    T = nst * c["dt"]
    assert abs(sig_num.real - sig.real) / abs(sig) < 1e-6
    dphase = (sig_num.imag - sig.imag) * T
    dphase = (dphase + np.pi) % (2 * np.pi) - np.pi
    assert abs(dphase) / T / abs(sig) < 1e-6
    assert abs(sig_num.real - gold.imag) / gold.imag < 1e-4
    ch.close()


def test_error_paths_on_device(B):
    c = inputs.config("cfg1")
    ch = B.Channel(c["nx"], c["ny"], c["nz"], c["lx"], c["lz"], c["y"], c["re"], c["dt"])
    with pytest.raises(B.ChanError) as e:
        ch.substep()
    assert e.value.status == B.ESTATE
    ch.bind("cuda:0")
    with pytest.raises(B.ChanError):
        ch.substep()                      # no state yet
    v, phi, omy = seeded_state(c)
    ch.set_state(v, phi, omy, c["U"], c["W"])
    ch.substep()
    with pytest.raises(B.ChanError) as e:
        ch.step()                         # mid-step
    assert e.value.status == B.ESTATE
    with pytest.raises(B.ChanError) as e:
        ch.filter_store(16, 3)            # kx cutoff beyond the retained range
    assert e.value.status == B.EINVAL
    small = torch.empty(10, dtype=torch.complex128, device="cuda")
    rc = ch.lib.chan_filter_store(ch.h, 2, 2, small.data_ptr(), small.numel() * 16)
    assert rc == B.ENOSPACE
    ch.close()


def test_host_buffer_entry_points(B):
    """The e2e path bench.py times: host state in, substeps, host state out."""
    c, ch, o = make(B, "cfg1")
    v, phi, omy = inputs.fluctuations(c)
    hv, hp, ho = (t.clone().pin_memory() for t in (v, phi, omy))
    hU, hW = torch.from_numpy(c["U"]).clone(), torch.from_numpy(c["W"]).clone()
    ch.set_state_host(hv, hp, ho, hU, hW)
    # chan.h: the call synchronises, the host buffers are the caller's again at once -- scribble on them
    for t in (hv, hp, ho, hU, hW):
        t.fill_(7.0)
    o.set_state(v.numpy(), phi.numpy(), omy.numpy(), c["U"], c["W"])
    ch.step()
    o.step()
    ch.get_state_host(hv, hp, ho, hU, hW)
    t = make_hp(o)
    t.set_state(v.numpy(), phi.numpy(), omy.numpy(), c["U"], c["W"])
    t.step()
    f = noise_floor(o, t)
    assert rel(hv, o.v) < 3 * TOL_SUBSTEP and rel(ho, o.omy) < max(3 * TOL_SUBSTEP, K_FLOOR * f["omy"])
    assert rel(hp, o.phi) < max(3 * TOL_SUBSTEP, K_FLOOR * f["phi"])
    out = torch.empty((10, c["ny"], 2 * 8 + 1, 9), dtype=torch.complex128).pin_memory()
    ch.filter_store_host(8, 8, out)
    assert rel(out, o.filter_store(8, 8)) < 1e-10
    ch.close()


def test_unlisted_transform_lengths_use_the_generic_kernels(B):
    """mx = 72, mz = 27: stage lists ([3,3|8], [3,3,3]) that have no compile-time specialisation, so the run-time
    radix-switch kernels (k_*_g) carry the planes; one full step, filter and statistics against the oracle."""
    c = inputs.config("cfg1", nx=48, nz=18, cut=(7, 5))
    ch = B.Channel(c["nx"], c["ny"], c["nz"], c["lx"], c["lz"], c["y"], c["re"], c["dt"]).bind("cuda:0")
    o = ChannelOracle(c["nx"], c["ny"], c["nz"], c["lx"], c["lz"], c["y"], c["re"], c["dt"])
    v, phi, omy = seeded_state(c, 20.0)
    ch.set_state(v, phi, omy, c["U"], c["W"])
    o.set_state(v, phi, omy, c["U"], c["W"])
    t = make_hp(o)
    t.set_state(v, phi, omy, c["U"], c["W"])
    ch.step()
    o.step()
    t.step()
    check_state(ch, o, t, 3, "generic")
    got = ch.filter_store(*c["cut"]).cpu().numpy()
    ref = o.filter_store(*c["cut"])
    for n in range(10):
        assert rel(got[n], ref[n]) < 1e-10, n
    ch.stats(B.STATS_RESET | B.STATS_ACCUMULATE)
    prof, _ = ch.stats(B.STATS_READ)
    assert np.abs(prof - o.stats_profiles()).max() < 1e-10 * np.abs(prof).max()
    ch.close()


def test_edge_sizes_smallest_grid_and_extreme_cutoffs(B):
    """Degenerate cases: the smallest grid the ABI accepts (ny = 8: every row of the compact operators is a wall or
    near-wall row; nx = 16, nz = 4: one tile, one-stage z transform), and the filter at its two extreme cutoffs
    (only the mean column / every retained mode)."""
    c = inputs.config("cfg2", ny=8, mesh=("cos", 0.5), dt=1e-3, re=100.0, mean=("poiseuille", 1.0), spec="gauss", M=3,
                      amp=("maxu", 1e-2), cut=(0, 0), seed=9)
    ch = B.Channel(c["nx"], c["ny"], c["nz"], c["lx"], c["lz"], c["y"], c["re"], c["dt"]).bind("cuda:0")
    o = ChannelOracle(c["nx"], c["ny"], c["nz"], c["lx"], c["lz"], c["y"], c["re"], c["dt"])
    v, phi, omy = seeded_state(c)
    ch.set_state(v, phi, omy, c["U"], c["W"])
    o.set_state(v, phi, omy, c["U"], c["W"])
    for n in range(3):
        ch.substep()
        o.substep()
    e = state_errors(ch, o)
    assert max(e["v"], e["phi"], e["omy"], e["U"]) < 3 * TOL_SUBSTEP, e
    for cut in ((0, 0), (c["nx"] // 2 - 1, c["nz"] // 2 - 1)):
        got = ch.filter_store(*cut).cpu().numpy()
        ref = o.filter_store(*cut)
        assert got.shape == ref.shape == (10, c["ny"], 2 * cut[1] + 1, cut[0] + 1)
        for n in range(10):
            assert rel(got[n], ref[n]) < 1e-10, (cut, n)
    with pytest.raises(B.ChanError) as ex:
        ch.filter_store(c["nx"] // 2, 0)          # one past the retained range
    assert ex.value.status == B.EINVAL
    ch.close()


def test_constant_pressure_gradient_forcing_and_narrow_stencils(B):
    """chan_opts_t: forcing = 1 (prescribed -dP/dx instead of the constant mass flux of PAPER.md L61) and the narrower
    compact schemes of reading R4 (half widths 2/2: the same kernels with zeros in the band tables)."""
    c = inputs.config("cfg1")
    v, phi, omy = seeded_state(c, 20.0)
    for forcing, hl, hr in ((1, 3, 3), (0, 2, 2)):
        ch = B.Channel(c["nx"], c["ny"], c["nz"], c["lx"], c["lz"], c["y"], c["re"], c["dt"], forcing=forcing, half_lhs=hl,
                       half_rhs=hr).bind("cuda:0")
        o = ChannelOracle(c["nx"], c["ny"], c["nz"], c["lx"], c["lz"], c["y"], c["re"], c["dt"], forcing=forcing, half_lhs=hl,
                          half_rhs=hr)
        ch.set_state(v, phi, omy, c["U"], c["W"])
        o.set_state(v, phi, omy, c["U"], c["W"])
        if forcing:
            ch.set_pgrad(1.25)
            o.pgrad = 1.25
        h = make_hp(o)                       # after pgrad: the yardstick copies the oracle's parameters
        h.set_state(v, phi, omy, c["U"], c["W"])
        for _ in range(3):
            ch.substep()
            o.substep()
            h.substep()
        e, f = check_state(ch, o, h, 3, (forcing, hl))
        assert max(e["v"], e["omy"], e["U"]) < 3 * TOL_SUBSTEP, (forcing, hl, e)
        assert ch.scalars()[0] == pytest.approx(o.pgrad, rel=1e-9)
        ch.close()


@pytest.mark.parametrize("name", ["cfg1", "mid"])
def test_step_filter_is_filter_store_then_step_bit_for_bit(B, name):
    """chan_step_filter: same database and same new state as the two separate calls."""
    c = inputs.config(name)
    v, phi, omy = seeded_state(c, 20.0 if name == "cfg1" else 1.0)
    outs = []
    for fused in (False, True):
        ch = B.Channel(c["nx"], c["ny"], c["nz"], c["lx"], c["lz"], c["y"], c["re"], c["dt"]).bind("cuda:0")
        ch.set_state(v, phi, omy, c["U"], c["W"])
        ch.step()
        if fused:
            db = ch.step_filter(*c["cut"])
        else:
            db = ch.filter_store(*c["cut"])
            ch.step()
        outs.append([db.clone()] + [t.clone() for t in ch.get_state()])
        if fused:
            ch.substep()
            with pytest.raises(B.ChanError) as ex:
                ch.step_filter(*c["cut"])         # mid-step
            assert ex.value.status == B.ESTATE
        ch.close()
    for a, b in zip(*outs):
        assert torch.equal(a, b)


@pytest.mark.parametrize("name,chunk_mb", [("mid", 3), ("cfg1", 0)])
def test_merged_plane_launches_equal_separate_launches(B, name, chunk_mb):
    """chan_tuning_t.plane_overlap: launch t of the merged kernel carries the inverse z pass of plane chunk t, the x pass
    of chunk t-1 and the forward z pass of chunk t-2 on double-buffered chunk buffers; the planes are independent, so
    the result must not depend on the launch structure or on the chunk size beyond rounding ("mid" with 3 MiB chunks:
    33 chunks of 2 planes against 17 chunks of 4, both with a ragged last one)."""
    c = inputs.config(name)
    v, phi, omy = seeded_state(c, 20.0 if name == "cfg1" else 1.0)
    res = []
    for overlap in (1, 2):
        ch = B.Channel(c["nx"], c["ny"], c["nz"], c["lx"], c["lz"], c["y"], c["re"], c["dt"],
                       tuning=dict(plane_overlap=overlap, chunk_mb=chunk_mb)).bind("cuda:0")
        t = ch.debug_get_tuning()
        assert t["plane_overlap"] == overlap
        if chunk_mb:
            assert 1 < t["planes_per_chunk"] < c["ny"] and c["ny"] % t["planes_per_chunk"] != 0
        ch.set_state(v, phi, omy, c["U"], c["W"])
        ch.step()
        db = ch.step_filter(*c["cut"])
        res.append([db.clone()] + [x.clone() for x in ch.get_state()] + [ch.debug_get_field(f) for f in (B.F_H1, B.F_H2, B.F_H3)])
        ch.close()
    # another kernel, another FMA contraction of the same source: equal to rounding, not bit for bit
    for a, b in zip(*res):
        assert rel(a, b.cpu().numpy()) < 1e-13


def _f32_close(got, ref, scale):
    """binary32 database against the oracle's: the two fp64 results differ by rounding (~1e-14 of the field's scale),
    so their roundings to binary32 agree to one unit in the last place of the component, plus that fp64 difference for
    components that are themselves far below the field's scale."""
    g = np.ascontiguousarray(got).view(np.float32).astype(np.float64)
    r = np.ascontiguousarray(ref).view(np.float32).astype(np.float64)
    lim = np.spacing(np.abs(ref.view(np.float32))).astype(np.float64) + 1e-13 * scale
    return bool((np.abs(g - r) <= lim).all()), float((np.abs(g - r) / lim).max())


def test_single_precision_database(B):
    """NEXT-1: chan_set_filter_precision(4) stores complex64 = the fp64 result rounded once to nearest
    even; the mode selection and everything upstream are unchanged."""
    c, ch, o = make(B, "cfg1")
    v, phi, omy = seeded_state(c, 20.0)
    ch.set_state(v, phi, omy, c["U"], c["W"])
    o.set_state(v, phi, omy, c["U"], c["W"])
    ch.step()
    o.step()
    kxc, kzc = c["cut"]
    d64 = ch.filter_store(kxc, kzc)
    ch.set_filter_precision(4)
    d32 = ch.filter_store(kxc, kzc)
    assert d32.dtype == torch.complex64 and d32.shape == d64.shape
    assert torch.equal(d32, d64.to(torch.complex64))                 # one rounding of the kernel's own fp64 value
    u = ch.debug_get_field(B.F_U).cpu().numpy()
    qs = [q % c["nz"] for q in list(range(0, kzc + 1)) + list(range(-kzc, 0))]
    assert np.array_equal(d32[0].cpu().numpy(), np.transpose(u[qs][:, : kxc + 1, :], (2, 0, 1)).astype(np.complex64))
    ref = o.filter_store(kxc, kzc, single=True)
    g = d32.cpu().numpy()
    for n in range(10):
        ok, worst = _f32_close(g[n], ref[n], float(np.abs(ref[n]).max()))
        assert ok, (n, worst)
    # fused into the step as well, and through the host entry point
    f32 = ch.step_filter(kxc, kzc)
    assert torch.equal(f32, d32)
    host = torch.empty(tuple(d32.shape), dtype=torch.complex64).pin_memory()
    ch.filter_store_host(kxc, kzc, host)
    o.step()
    assert _f32_close(host.numpy()[4], o.filter_store(kxc, kzc, single=True)[4], float(np.abs(ref[4]).max()))[0]
    small = torch.empty(d32.numel() - 1, dtype=torch.complex64, device="cuda")
    assert ch.lib.chan_filter_store(ch.h, kxc, kzc, small.data_ptr(), small.numel() * 8) == B.ENOSPACE
    assert ch.lib.chan_set_filter_precision(ch.h, 5) == B.EINVAL
    ch.close()


@pytest.mark.parametrize("single", [False, True])
def test_run_cadence_equals_the_calls_written_out(B, single):
    """NEXT-1: chan_run(nsteps, filter_every, stats_every) == the same chan_stats /
    chan_step_filter / chan_step calls issued one by one (bit for bit: same kernels), and == oracle.run."""
    c = inputs.config("cfg1")
    v, phi, omy = seeded_state(c, 20.0)
    kxc, kzc = c["cut"]
    a = B.Channel(c["nx"], c["ny"], c["nz"], c["lx"], c["lz"], c["y"], c["re"], c["dt"]).bind("cuda:0")
    b = B.Channel(c["nx"], c["ny"], c["nz"], c["lx"], c["lz"], c["y"], c["re"], c["dt"]).bind("cuda:0")
    o = ChannelOracle(c["nx"], c["ny"], c["nz"], c["lx"], c["lz"], c["y"], c["re"], c["dt"])
    for x in (a, b, o):
        x.set_state(v, phi, omy, c["U"], c["W"])
    if single:
        a.set_filter_precision(4)
        b.set_filter_precision(4)
    ring, n = a.run(5, 2, 1, kxc, kzc)
    assert n == 3 and ring.shape[0] == 3
    want = []
    b.stats(B.STATS_RESET)
    for k in range(5):
        b.stats(B.STATS_ACCUMULATE)
        if k % 2 == 0:
            want.append(b.step_filter(kxc, kzc).clone())
        else:
            b.step()
    for k in range(3):
        assert torch.equal(ring[k], want[k]), k
    for x, y in zip(a.get_state(), b.get_state()):
        assert torch.equal(x, y)
    sa, na = a.stats(B.STATS_READ)
    sb, nb = b.stats(B.STATS_READ)
    assert na == nb == 5
    if single:
        assert np.array_equal(sa, sb)                  # binary32 database: the statistics keep their own pass
    else:                                              # fp64 database: taken from its (0,0) modes on the emitting steps
        assert np.abs(sa - sb).max() < 1e-13 * np.abs(sb).max()
    snaps = o.run(5, 2, 1, kxc, kzc, single=single)
    so, no = o.stats_read()
    assert no == 5 and np.abs(sa - so).max() < 1e-10 * np.abs(so).max()
    for k in range(3):
        g = ring[k].cpu().numpy()
        for m in range(10):
            if single:
                ok, worst = _f32_close(g[m], snaps[k][m], float(np.abs(snaps[k][m]).max()))
                assert ok, (k, m, worst)
            else:
                assert rel(g[m], snaps[k][m]) < 1e-10, (k, m)
    # a ring of two slots wraps: the third snapshot lands in slot 0
    a.set_state(v, phi, omy, c["U"], c["W"])
    ring2, n2 = a.run(5, 2, 0, kxc, kzc, ring_slots=2)
    assert n2 == 3 and torch.equal(ring2[0], want[2]) and torch.equal(ring2[1], want[1])
    # error paths
    a.substep()
    r = B.Run(1, 1, 0, kxc, kzc, ring2.data_ptr(), ring2[0].numel() * ring2.element_size(), 2)
    assert a.lib.chan_run(a.h, r, None) == B.ESTATE                       # mid-step
    a.substep()
    a.substep()
    r.slot_bytes = 16
    assert a.lib.chan_run(a.h, r, None) == B.ENOSPACE
    r.dev_ring = None
    assert a.lib.chan_run(a.h, r, None) == B.EINVAL
    a.close()
    b.close()


def test_postprocessing_of_the_stored_database(B):
    """NEXT-2: filtered pressure (3.2), strain norm (3.3 as re-derived, R17) and sub-grid stresses
    (3.4) computed by the library from a database it wrote, against oracle/postprocess.py on the same database; once
    with the handle that ran the flow and once with a small handle on the storage grid (offline post-processing)."""
    from oracle.postprocess import DatabaseOracle
    c, ch, o = make(B, "mid")
    v, phi, omy = seeded_state(c)
    ch.set_state(v, phi, omy, c["U"], c["W"])
    ch.step()
    kxc, kzc = c["cut"]
    db = ch.filter_store(kxc, kzc)
    dbn = db.cpu().numpy()
    po = DatabaseOracle(o.y, o.lx, o.lz, kxc, kzc, o.nu, o.A1, o.B1, o.A2, o.B2)
    p_ref, s_ref, t_ref = po.filtered_pressure(dbn), po.strain_norm(dbn), po.sgs_tensor(dbn)
    state0 = [t.clone() for t in ch.get_state()]
    derived0 = [ch.debug_get_field(f).clone() for f in (B.F_U, B.F_W, B.F_OMX, B.F_OMZ)]
    # storage-grid handle: nx >= 2 (Kx + 1), nz >= 2 (Kz + 1) with admissible transform lengths
    small = B.Channel(32, c["ny"], 16, c["lx"], c["lz"], c["y"], c["re"], c["dt"]).bind("cuda:0")
    for hnd, name in ((ch, "flow handle"), (small, "storage-grid handle")):
        p = hnd.post_pressure(kxc, kzc, db).cpu().numpy()
        live = np.ones(p.shape[1:], bool)
        assert rel(p, p_ref) < 1e-9, (name, rel(p, p_ref))
        assert rel(hnd.post_strain_norm(kxc, kzc, db), s_ref) < 1e-12, name
        tau = hnd.post_sgs(kxc, kzc, db).cpu().numpy()
        for n in range(6):
            assert np.abs(tau[n] - t_ref[n]).max() < 1e-12 * max(1.0, np.abs(dbn[3 + n]).max()), (name, n)
    small.close()
    # the flow handle is unchanged by the post-processing calls: state untouched, derived fields rebuilt bit for bit
    for a, b in zip(state0, ch.get_state()):
        assert torch.equal(a, b)
    for a, f in zip(derived0, (B.F_U, B.F_W, B.F_OMX, B.F_OMZ)):
        assert torch.equal(a, ch.debug_get_field(f))
    # error paths
    scratch = torch.empty(64, dtype=torch.uint8, device="cuda")
    out = torch.empty_like(db[0])
    assert ch.lib.chan_post_pressure(ch.h, kxc, kzc, db.data_ptr(), out.data_ptr(), scratch.data_ptr(), 64) == B.ENOSPACE
    assert ch.lib.chan_post_scratch_bytes(ch.h, c["nx"], 0) == 0
    ch.substep()
    n = int(ch.lib.chan_post_scratch_bytes(ch.h, kxc, kzc))
    big = torch.empty(n, dtype=torch.uint8, device="cuda")
    tau = torch.empty((6,) + tuple(db.shape[1:]), dtype=torch.complex128, device="cuda")
    assert ch.lib.chan_post_sgs(ch.h, kxc, kzc, db.data_ptr(), tau.data_ptr(), big.data_ptr(), n) == B.ESTATE    # mid-step
    ch.close()


@pytest.mark.parametrize("name,tz", [("mid", 8), ("cfg1", 4)])
def test_cluster_z_passes_equal_single_cta_z_passes(B, name, tz):
    """chan_tuning_t.z_cluster: the z tile split by rows over a 2-CTA cluster (the first inverse / last forward stage
    exchanges half of its data through distributed shared memory) against one CTA per tile: a step, the fused filter
    (ragged last tile: the filter's 12 columns in tiles of 16 on "mid") and the nonlinear term, equal to rounding."""
    c = inputs.config(name)
    v, phi, omy = seeded_state(c, 20.0 if name == "cfg1" else 1.0)
    res = []
    for zc in (1, 2):
        ch = B.Channel(c["nx"], c["ny"], c["nz"], c["lx"], c["lz"], c["y"], c["re"], c["dt"], tuning=dict(z_cluster=zc, tz=tz)).bind("cuda:0")
        t = ch.debug_get_tuning()
        assert t["z_cluster"] == zc and t["tz"] == (2 * tz if zc == 2 else tz)
        ch.set_state(v, phi, omy, c["U"], c["W"])
        ch.step()
        db = ch.step_filter(*c["cut"])
        res.append([db.clone()] + [x.clone() for x in ch.get_state()] + [ch.debug_get_field(f) for f in (B.F_H1, B.F_H2, B.F_H3)])
        ch.close()
    for a, b in zip(*res):
        assert rel(a, b.cpu().numpy()) < 1e-13


@pytest.mark.parametrize("name", ["cfg1", "mid"])
def test_spectra(B, name):
    """chan_spectra (NEXT-4) against oracle.spectra, and its consistency with chan_stats."""
    c, ch, o = make(B, name)
    v, phi, omy = seeded_state(c, 20.0 if name == "cfg1" else 1.0)
    ch.set_state(v, phi, omy, c["U"], c["W"])
    o.set_state(v, phi, omy, c["U"], c["W"])
    ch.step()
    o.step()
    ex, ez = (t.cpu().numpy() for t in ch.spectra())
    rx, rz = o.spectra()
    for n in range(7):
        assert np.abs(ex[n] - rx[n]).max() < 1e-10 * np.abs(rx[n]).max(), n
        assert np.abs(ez[n] - rz[n]).max() < 1e-10 * np.abs(rz[n]).max(), n
    ch.stats(B.STATS_RESET | B.STATS_ACCUMULATE)
    prof, _ = ch.stats(B.STATS_READ)
    for n in range(7):
        sc = max(1.0, np.abs(prof[3 + n]).max())
        assert np.abs(ex[n].sum(axis=1) - prof[3 + n]).max() < 1e-12 * sc and np.abs(ez[n].sum(axis=1) - prof[3 + n]).max() < 1e-12 * sc
    small = torch.empty(8, dtype=torch.float64, device="cuda")
    assert ch.lib.chan_spectra(ch.h, small.data_ptr(), 64, None, 0) == B.ENOSPACE
    assert ch.lib.chan_spectra(ch.h, None, 0, None, 0) == B.EINVAL
    ch.close()
