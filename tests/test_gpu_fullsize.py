"""GPU parity at BASELINE.json's full sizes, in the launch configuration bench.py times (same plans, tiles, chunking).

The oracle cannot run a 768x251x576 (or larger) substep in seconds, but every stage of the path is separable:
the wall-normal stages act on each (kx,kz) line independently and the wall-parallel stages on each y-plane
independently.  So the full-size GPU result is compared with the oracle on SAMPLED lines and planes:

* lines: a small ChannelOracle on the same mesh whose wavenumber tables are overwritten with those of a
  64 x 64 sub-lattice {p} x {z slot} of the big grid (4096 lines, including the mean mode and the z-Nyquist slot)
  computes exactly those lines of the big problem; the long-double yardstick (oracle/channel_hp.py) runs on a
  16 x 16 sub-lattice of those and gives the oracle's own rounding error, which sets the gate where it exceeds
  north_star's 1e-11;
* planes: a ChannelOracle with the full nx, nz runs the padded transforms, the products, the filter products and
  the statistics of 64 sampled planes (in batches of 8), among them both sides of the first, a middle and the last
  plane-chunk seam of the launch configuration (chan_debug_get_tuning: planes_per_chunk).

All inputs are seeded; the oracle receives copies of the very arrays handed to the library.
"""
import copy
import os

import numpy as np
import pytest
import torch

import __graft_entry__ as entry
from oracle.channel import ChannelOracle
from paper_1808_06461_b200 import inputs
from test_gpu_parity import K_FLOOR, K_LINE, line_rel, make_hp, rel

pytestmark = pytest.mark.gpu

TOL_SUBSTEP = 1e-11


@pytest.fixture(scope="module")
def B():
    if not torch.cuda.is_available():
        pytest.skip("no CUDA device")
    entry.build()
    from paper_1808_06461_b200 import binding
    return binding


def sub_lattice(c, npx=64, nsz=64):
    """Index lists (p, z slot) of the sampled lines; entry [0] of each is 0 (mean mode) and the middle z entry is
    the Nyquist slot, so the small oracle's special cases coincide with the big grid's."""
    nxh, nz = c["nx"] // 2, c["nz"]
    rng = np.random.default_rng(11)
    ps = np.sort(np.concatenate([[0, 1, nxh - 1], rng.choice(np.arange(2, nxh - 1), npx - 3, replace=False)]))
    lo = np.sort(np.concatenate([[0, 1], rng.choice(np.arange(2, nz // 2), nsz // 2 - 2, replace=False)]))
    hi = np.sort(np.concatenate([[nz - 1], rng.choice(np.arange(nz // 2 + 1, nz - 1), nsz // 2 - 2, replace=False)]))
    ss = np.concatenate([lo, [nz // 2], hi])
    assert ps.size == npx and ss.size == nsz and ss[nsz // 2] == nz // 2
    return ps, ss


def line_oracle(c, ps, ss, cls=ChannelOracle):
    from oracle.channel import wavenumbers
    kx, kz, _ = wavenumbers(c["nx"], c["nz"], c["lx"], c["lz"])
    o = cls(2 * ps.size, c["ny"], ss.size, c["lx"], c["lz"], c["y"], c["re"], c["dt"])
    o.kx, o.kz = kx[ps].copy(), kz[ss].copy()
    o.k2 = o.kz[:, None] ** 2 + o.kx[None, :] ** 2
    return o


HP_STRIDE = 4      # the long-double yardstick runs on every 4th p and z slot of the sub-lattice (16 x 16 lines)


def sub_oracle(base, ps, ss, ip, iz):
    """The oracle restricted to the lines (ss[iz], ps[ip]) of `base` (which already carries the sampled wavenumbers):
    same tables (built once in exact rationals), fresh state.  iz must keep 0 first and the Nyquist slot in the middle."""
    o = copy.copy(base)
    o.nx, o.nz = 2 * len(ip), len(iz)
    o.mx, o.mz = 3 * o.nx // 2, 3 * o.nz // 2
    o.kx, o.kz = base.kx[ip].copy(), base.kz[iz].copy()
    o.k2 = o.kz[:, None] ** 2 + o.kx[None, :] ** 2
    shp = (o.nz, o.nx // 2, o.ny)
    o.v, o.phi, o.omy, o.hv_prev, o.hg_prev = (np.zeros(shp, complex) for _ in range(5))
    o.U, o.W, o.H1m_prev, o.H3m_prev = (np.zeros(o.ny) for _ in range(4))
    return o


def hp_indices(ps, ss):
    ip, iz = np.arange(0, ps.size, HP_STRIDE), np.arange(0, ss.size, HP_STRIDE)
    assert ip[0] == 0 and iz[0] == 0 and iz[iz.size // 2] == ss.size // 2      # mean mode and Nyquist slot stay in place
    return ip, iz


def ysolve_reference(base, ps, ss, state, Hl, isub, c):
    """Oracle on all sampled lines and long-double yardstick on the 16 x 16 subset, for one substep coefficient set from
    seeded H and history.  Returns (oracle, subset oracle, yardstick, subset index arrays)."""
    sv, sphi, somy = state
    o = copy.deepcopy(base)
    o.set_state(sv, sphi, somy, c["U"], c["W"])
    o.isub = isub
    o.hv_prev, o.hg_prev = Hl[3].copy(), Hl[4].copy()
    o.nonlinear = lambda fields: tuple(h.copy() for h in Hl[:3])
    o.substep()
    ip, iz = hp_indices(ps, ss)
    pick = lambda a: a[np.ix_(iz, ip)]
    os_ = sub_oracle(base, ps, ss, ip, iz)
    hp = make_hp(os_)
    for orc in (os_, hp):
        orc.set_state(pick(sv), pick(sphi), pick(somy), c["U"], c["W"])
        orc.isub = isub
        orc.hv_prev, orc.hg_prev = pick(Hl[3]).astype(orc.v.dtype), pick(Hl[4]).astype(orc.v.dtype)
    os_.nonlinear = lambda fields: tuple(pick(h).copy() for h in Hl[:3])
    hp.nonlinear_override = lambda fields: tuple(pick(h) for h in Hl[:3])
    os_.substep()
    hp.substep()
    # the subset oracle is the big one restricted (same arithmetic per line): bit for bit
    assert np.array_equal(os_.phi, pick(o.phi)) and np.array_equal(os_.v, pick(o.v))
    return o, os_, hp, (ip, iz)


def gate_ysolve(name, isub, gpu, o, os_, hp, sub):
    """gpu = (v, phi, om_y lines [64][64][ny], U).  Whole-sample relative L2 and per-line gates."""
    ip, iz = sub
    pick = lambda a: a[np.ix_(iz, ip)]
    e, fl, eh = {}, {}, {}
    for k, g in zip(("v", "phi", "omy"), gpu[:3]):
        ref = getattr(o, k)
        hpk = np.asarray(getattr(hp, k)).astype(complex)
        e[k] = rel(g, ref)
        fl[k] = rel(getattr(os_, k), hpk)                 # oracle's own rounding error (16 x 16 lines)
        eh[k] = rel(pick(g), hpk)                         # kernel's rounding error on the same lines
    e["U"], fl["U"], eh["U"] = rel(gpu[3], o.U), rel(os_.U, np.asarray(hp.U).astype(float)), rel(gpu[3], np.asarray(hp.U).astype(float))
    print(f"{name} substep set {isub}: |gpu-oracle| {e}  |oracle-hp| {fl}  |gpu-hp| {eh}")
    for k in e:
        lim = max(TOL_SUBSTEP, K_FLOOR * fl[k])
        assert e[k] < lim and eh[k] < lim, (isub, k, e, fl, eh)
    assert max(e["v"], e["U"]) < TOL_SUBSTEP, (isub, e)    # the primitive unknowns meet north_star outright
    # per line: all 4096 against the oracle, bound = the worst oracle rounding error among the yardstick's lines
    for k, g in zip(("v", "phi", "omy"), gpu[:3]):
        ref = getattr(o, k)
        el = line_rel(g, ref)
        fworst = float(line_rel(np.asarray(getattr(hp, k)).astype(complex), getattr(os_, k)).max())
        assert el.max() < max(TOL_SUBSTEP, K_LINE * fworst), (isub, k, "line", np.unravel_index(np.argmax(el), el.shape), float(el.max()), fworst)


def sample_planes(ny, pc, n=64):
    """n plane indices: the walls and their neighbours, both sides of the first, a middle and the last chunk seam
    (chunks are [k pc, (k+1) pc)), the rest spread over y."""
    must = {0, 1, 2, ny - 3, ny - 2, ny - 1, ny // 2}
    nch = (ny + pc - 1) // pc
    for k in {1, nch // 2, nch - 1}:
        if 0 < k < nch:
            must |= {k * pc - 1, k * pc}
    must = {j for j in must if 0 <= j < ny}
    rng = np.random.default_rng(17)
    rest = rng.permutation(np.setdiff1d(np.arange(ny), sorted(must)))[: max(0, min(n, ny) - len(must))]
    return sorted(must | set(int(j) for j in rest))


def planes_check(B, ch, c, planes, sampled, nonlinear=True):
    """a13, a14, a3-a8 on the sampled planes against the oracle, in batches of 8 planes.  sampled: six numpy arrays
    [nz][nxh][len(planes)] = the seeded fields on those planes."""
    nz = c["nz"]
    kxc, kzc = c["cut"]
    got = ch.filter_store(kxc, kzc)
    gp = got[:, planes].cpu().numpy()
    del got
    slots = [q % nz for q in list(range(0, kzc + 1)) + list(range(-kzc, 0))]
    for n in range(3):
        assert np.array_equal(gp[n], np.transpose(sampled[n][slots][:, : kxc + 1, :], (2, 0, 1))), n
    ch.stats(B.STATS_RESET | B.STATS_ACCUMULATE)
    prof, ns = ch.stats(B.STATS_READ)
    assert ns == 1
    wp = np.full(c["nx"] // 2, 2.0)
    wp[0] = 1.0
    mean = lambda a, b: np.einsum("p,qpy->y", wp, (a * np.conj(b)).real)
    u, v, w, ox, oy, oz = sampled
    ref = [u[0, 0].real, v[0, 0].real, w[0, 0].real, mean(u, u), mean(u, v), mean(u, w), mean(v, v), mean(v, w), mean(w, w),
           mean(ox, ox) + mean(oy, oy) + mean(oz, oz)]
    for n in range(10):
        assert np.abs(prof[n][planes] - ref[n]).max() < 1e-12 * max(1.0, np.abs(ref[n]).max()), n
    for n in range(3, 10):   # second-order consistency on the GPU side: (0,0) mode of the stored products == statistics
        assert np.abs(gp[n][:, 0, 0].real - prof[n][planes]).max() < 1e-11 * np.abs(prof[n]).max()
    H = None
    if nonlinear:
        ch.debug_run_stage(B.STAGE_NONLINEAR)
        H = []
        for fid in (B.F_H1, B.F_H2, B.F_H3):
            g = ch.debug_get_field(fid)
            assert not bool(g[nz // 2].any())
            H.append(g[:, :, planes].cpu().numpy())
            del g
    nb = 8
    o = ChannelOracle(c["nx"], nb, nz, c["lx"], c["lz"], np.linspace(-1, 1, nb), c["re"], c["dt"])
    worst = 0.0
    for b0 in range(0, len(planes), nb):
        sl = slice(b0, min(b0 + nb, len(planes)))
        cnt = sl.stop - sl.start
        batch = []
        for f in sampled:                       # pad the last batch with zero planes: the oracle is built for nb planes
            a = np.zeros(f.shape[:2] + (nb,), complex)
            a[:, :, :cnt] = f[:, :, sl]
            batch.append(a)
        pu, pv, pw, pox, poy, poz = (o.to_physical(f) for f in batch)
        prods = (pu * pu, pu * pv, pu * pw, pv * pv, pv * pw, pw * pw, pox * pox + poy * poy + poz * poz)
        for n, pr in enumerate(prods):
            r = rel(gp[3 + n][sl], o.to_spectral(pr, kxc, kzc)[:cnt])
            worst = max(worst, r)
            assert r < 1e-13, (n, b0)
        if nonlinear:
            refs = (o.to_spectral(pv * poz - pw * poy), o.to_spectral(pw * pox - pu * poz), o.to_spectral(pu * poy - pv * pox))
            for g, ref_h in zip(H, refs):
                r = rel(g[:, :, sl], ref_h[:, :, :cnt])
                worst = max(worst, r)
                assert r < 1e-13, b0
    print(f"planes {len(planes)} (seams included): worst relative L2 of a batch of 8 planes {worst:.2e}")


def take_lines(t, ps, ss):
    """[nz][nxh][ny] torch tensor (any device) -> numpy [len(ss)][len(ps)][ny]."""
    idx_s = torch.as_tensor(ss, device=t.device)
    idx_p = torch.as_tensor(ps, device=t.device)
    return t.index_select(0, idx_s).index_select(1, idx_p).cpu().numpy()


def random_field(shape, nz, seed, dev, scale=1.0):
    g = torch.Generator(device=dev).manual_seed(seed)
    r = torch.randn(shape + (2,), generator=g, dtype=torch.float64, device=dev)
    if scale != 1.0:
        r.mul_(scale)                            # in place: config 5 leaves room for one 14.5 GB temporary only
    f = torch.view_as_complex(r)
    q = torch.arange(1, nz // 2, device=dev)
    f[nz - q, 0] = torch.conj(f[q, 0])          # Hermitian p = 0 column
    f[0, 0] = f[0, 0].real + 0j
    f[nz // 2] = 0
    return f


def _skip_if_whole_config5_fits():
    """The "cfg5-planes" / "cfg5-lines" cases exercise the plane size and the line length of config 5 on a fraction of its
    memory; where the device holds the whole config (test_config5_whole_on_sampled_lines_and_planes) they repeat it."""
    import gc
    gc.collect()
    torch.cuda.empty_cache()
    if torch.cuda.mem_get_info(0)[0] >= 170e9 and "cfg5" in (os.environ.get("CHAN_TEST_FULLSIZE") or "cfg5").split(","):
        pytest.skip("covered by test_config5_whole_on_sampled_lines_and_planes on this device")


def fullsize_names():
    """cfg3 and cfg4 by default (about 90 s together); CHAN_TEST_FULLSIZE=cfg3[,cfg4][,cfg5] restricts the list.
    Config 5 has a memory-lean test of its own below (its 148 GB workspace leaves room for one full-size field at a
    time) plus the cheap "cfg5-planes" / "cfg5-lines" cases."""
    env = os.environ.get("CHAN_TEST_FULLSIZE")
    return [n for n in env.split(",") if n in ("cfg3", "cfg4")] if env else ["cfg3", "cfg4"]


@pytest.mark.parametrize("name", fullsize_names() + ["cfg5-planes"])
def test_fullsize_planes_filter_stats(B, name):
    """a3-a8, a13, a14 at full size on 64 sampled planes (chunk seams included), from six seeded random Hermitian
    fields.  "cfg5-planes": the 1536 x 1152 wall-parallel grid of config 5 (its transform plans and tiles) on 72 planes
    with the plane chunks cut down to 11 planes as in the full config 5, so that the seams exist."""
    if name == "cfg5-planes":
        _skip_if_whole_config5_fits()
        c = inputs.config("cfg5", ny=72)
        tuning = None            # 3 GB chunks = 11 planes of this plane size, as in the full config
    else:
        c, tuning = inputs.config(name), None
    dev = torch.device("cuda:0")
    ch = B.Channel(c["nx"], c["ny"], c["nz"], c["lx"], c["lz"], c["y"], c["re"], c["dt"], tuning=tuning).bind(dev)
    nz, ny = c["nz"], c["ny"]
    pc = ch.debug_get_tuning()["planes_per_chunk"]
    planes = sample_planes(ny, pc)
    assert len(planes) == min(64, ny) and (pc >= ny or {pc - 1, pc} <= set(planes))
    fids = (B.F_U, B.F_V, B.F_W, B.F_OMX, B.F_OMY, B.F_OMZ)
    z = torch.zeros(ch.shape, dtype=torch.complex128, device=dev)
    ch.set_state(z, z, z, c["U"], c["W"])       # the filter and the statistics want a state; the six fields are overwritten below
    ch._keep = None
    del z
    sampled = []
    for k, fid in enumerate(fids):
        f = random_field(ch.shape, nz, 1000 + k, dev)
        ch.debug_set_field(fid, f)
        sampled.append(f[:, :, planes].cpu().numpy())
        del f
    torch.cuda.empty_cache()
    planes_check(B, ch, c, planes, sampled)
    ch.close()


@pytest.mark.parametrize("name", fullsize_names() + ["cfg5-lines"])
def test_fullsize_lines_derive_and_ysolve(B, name):
    """a1-a2 and a9-a12 at full size on 4096 sampled lines, for the three substep coefficient sets.
    "cfg5-lines": the 1025-point mesh, Re and dt of config 5 on a 128 x 64 sub-box with the same dx, dz (the same
    range of wavenumbers and Helmholtz parameters, the full line length, every line sampled)."""
    if name == "cfg5-lines":
        _skip_if_whole_config5_fits()
        c5 = inputs.CONFIGS["cfg5"]
        c = inputs.config("cfg5", nx=128, nz=64, lx=c5["lx"] * 128 / c5["nx"], lz=c5["lz"] * 64 / c5["nz"])
        ps, ss = np.arange(64), np.arange(64)
    else:
        c = inputs.config(name)
        ps, ss = sub_lattice(c)
    dev = torch.device("cuda:0")
    ch = B.Channel(c["nx"], c["ny"], c["nz"], c["lx"], c["lz"], c["y"], c["re"], c["dt"]).bind(dev)
    nz = c["nz"]
    v, phi, omy = inputs.fluctuations(c, device=dev, zchunk=64)
    state = tuple(take_lines(t, ps, ss) for t in (v, phi, omy))
    ch.set_state(v, phi, omy, c["U"], c["W"])
    del v, phi, omy
    ch._keep = None
    torch.cuda.empty_cache()
    base = line_oracle(c, ps, ss)
    o = copy.deepcopy(base)
    o.set_state(*state, c["U"], c["W"])
    # a1-a2
    refs = o.velocities_vorticities()
    for fid, ref in zip((B.F_U, B.F_V, B.F_W, B.F_OMX, B.F_OMY, B.F_OMZ), refs):
        g = ch.debug_get_field(fid)
        assert rel(take_lines(g, ps, ss), ref) < 1e-12, fid
        del g
    # a9-a12 with seeded H and history
    Hs, Hl = [], []
    for k, fid in enumerate((B.F_H1, B.F_H2, B.F_H3, B.F_HV_PREV, B.F_HG_PREV)):
        f = random_field(ch.shape, nz, 2000 + k, dev, scale=1e2 if k < 3 else 1.0)
        if k >= 3:
            f[0, 0] = 0
        Hl.append(take_lines(f, ps, ss))
        Hs.append(f)
    for isub in range(3):
        o, os_, hp, sub = ysolve_reference(base, ps, ss, state, Hl, isub, c)
        v, phi, omy = inputs.fluctuations(c, device=dev, zchunk=64)
        ch.set_state(v, phi, omy, c["U"], c["W"])
        del v, phi, omy
        ch._keep = None
        for f, fid in zip(Hs, (B.F_H1, B.F_H2, B.F_H3, B.F_HV_PREV, B.F_HG_PREV)):
            ch.debug_set_field(fid, f)
        ch.debug_set_substep_index(isub)
        ch.debug_run_stage(B.STAGE_YSOLVE)
        gv, gphi, gomy, gU, gW = ch.get_state()
        gpu = (take_lines(gv, ps, ss), take_lines(gphi, ps, ss), take_lines(gomy, ps, ss), gU.cpu().numpy())
        del gv, gphi, gomy
        gate_ysolve(name, isub, gpu, o, os_, hp, sub)
        assert rel(take_lines(ch.debug_get_field(B.F_HV_PREV), ps, ss), o.hv_prev) < 1e-11
        assert rel(take_lines(ch.debug_get_field(B.F_HG_PREV), ps, ss), o.hg_prev) < 1e-13
        # the new state's derived fields (a1 chained behind the y-solve) on the same lines
        ch.debug_run_stage(B.STAGE_DERIVE)
        refs = o.velocities_vorticities()
        for fid, ref in zip((B.F_U, B.F_W, B.F_OMX, B.F_OMZ), (refs[0], refs[2], refs[3], refs[5])):
            assert rel(take_lines(ch.debug_get_field(fid), ps, ss), ref) < 1e-8, fid
    ch.close()


def test_config5_whole_on_sampled_lines_and_planes(B):
    """The full 1536 x 1025 x 1152 config 5 in bench.py's launch configuration.  Memory-lean variant of the two tests
    above: the state is staged in host memory (chan_set_state_host), every other full-size field lives on the device
    one at a time and is regenerated from its seed when it is needed again.  4096 lines, all three substep
    coefficient sets; 64 planes with the chunk seams."""
    env = os.environ.get("CHAN_TEST_FULLSIZE")
    if env and "cfg5" not in env.split(","):
        pytest.skip("CHAN_TEST_FULLSIZE excludes cfg5")
    c = inputs.config("cfg5")
    dev = torch.device("cuda:0")
    nz, ny = c["nz"], c["ny"]
    shape = (nz, c["nx"] // 2, ny)
    import gc
    gc.collect()
    torch.cuda.empty_cache()
    free = torch.cuda.mem_get_info(dev)[0]
    if free < 166e9:
        pytest.skip(f"config 5 needs its 148 GB workspace plus one 14.5 GB field and the filter output on the device ({free / 1e9:.1f} GB free, "
                    f"{torch.cuda.memory_allocated(dev) / 1e9:.1f} GB allocated / {torch.cuda.memory_reserved(dev) / 1e9:.1f} GB reserved by this process)")
    hv, hp_, ho = (torch.empty(shape, dtype=torch.complex128) for _ in range(3))
    inputs.fluctuations(c, device=dev, zchunk=16, out=(hv, hp_, ho))
    hU, hW = torch.from_numpy(c["U"]).clone(), torch.from_numpy(c["W"]).clone()
    torch.cuda.empty_cache()
    ch = B.Channel(c["nx"], ny, nz, c["lx"], c["lz"], c["y"], c["re"], c["dt"]).bind(dev)
    ps, ss = sub_lattice(c)
    state = tuple(take_lines(t, ps, ss) for t in (hv, hp_, ho))
    base = line_oracle(c, ps, ss)

    def gpu_lines(fid):
        g = ch.debug_get_field(fid)
        out = take_lines(g, ps, ss)
        del g
        return out

    # ---- lines: a1-a2, then a9-a12 for the three substep coefficient sets
    ch.set_state_host(hv, hp_, ho, hU, hW)
    o = copy.deepcopy(base)
    o.set_state(*state, c["U"], c["W"])
    for fid, ref in zip((B.F_U, B.F_V, B.F_W, B.F_OMX, B.F_OMY, B.F_OMZ), o.velocities_vorticities()):
        assert rel(gpu_lines(fid), ref) < 1e-12, fid
    fids = (B.F_H1, B.F_H2, B.F_H3, B.F_HV_PREV, B.F_HG_PREV)
    for isub in (0, 1, 2):
        ch.set_state_host(hv, hp_, ho, hU, hW)
        Hl = []
        for k, fid in enumerate(fids):
            f = random_field(shape, nz, 2000 + k, dev, scale=1e2 if k < 3 else 1.0)
            if k >= 3:
                f[0, 0] = 0
            Hl.append(take_lines(f, ps, ss))
            ch.debug_set_field(fid, f)
            del f
            torch.cuda.empty_cache()
        o, os_, hp, sub = ysolve_reference(base, ps, ss, state, Hl, isub, c)
        ch.debug_set_substep_index(isub)
        ch.debug_run_stage(B.STAGE_YSOLVE)
        gl = [gpu_lines(B.F_V), gpu_lines(B.F_PHI), gpu_lines(B.F_OMY)]
        ch.debug_run_stage(B.STAGE_DERIVE)
        ch.stats(B.STATS_RESET | B.STATS_ACCUMULATE)
        prof, _ = ch.stats(B.STATS_READ)
        gate_ysolve("cfg5", isub, (*gl, prof[0]), o, os_, hp, sub)        # <u>(y) is the mean profile
    # ---- planes: filter, statistics, nonlinear term from six seeded random fields
    planes = sample_planes(ny, ch.debug_get_tuning()["planes_per_chunk"])
    sampled = []
    for k, fid in enumerate((B.F_U, B.F_V, B.F_W, B.F_OMX, B.F_OMY, B.F_OMZ)):
        f = random_field(shape, nz, 1000 + k, dev)
        ch.debug_set_field(fid, f)
        sampled.append(f[:, :, planes].cpu().numpy())
        del f
        torch.cuda.empty_cache()
    planes_check(B, ch, c, planes, sampled)
    ch.close()


@pytest.mark.parametrize("name", ["cfg3", "cfg4"])
def test_fullsize_chained_substep_equals_the_staged_one(B, name):
    """Property at full size: chan_substep hands D1-forward(v) from the last y sweep straight to the a1 sweeps; running
    the three stages one by one through the debug hooks recomputes it from the stored v.  Both must give the same
    fields bit for bit (the stages themselves are checked against the oracle above).  Config 4 has several plane chunks
    with a ragged last one."""
    c = inputs.config(name)
    dev = torch.device("cuda:0")
    v, phi, omy = inputs.fluctuations(c, device=dev, zchunk=64)
    hv, hphi, homy = v.cpu(), phi.cpu(), omy.cpu()
    del v, phi, omy
    res = []
    fields = (B.F_V, B.F_PHI, B.F_OMY, B.F_U, B.F_W, B.F_OMX, B.F_OMZ)
    for chained in (True, False):
        torch.cuda.empty_cache()
        ch = B.Channel(c["nx"], c["ny"], c["nz"], c["lx"], c["lz"], c["y"], c["re"], c["dt"]).bind(dev)
        ch.set_state_host(hv, hphi, homy, torch.from_numpy(c["U"]).clone(), torch.from_numpy(c["W"]).clone())
        if chained:
            ch.substep()
        else:
            ch.debug_run_stage(B.STAGE_NONLINEAR)
            ch.debug_run_stage(B.STAGE_YSOLVE)
            ch.debug_run_stage(B.STAGE_DERIVE)
        out = []
        for f in fields:
            g = ch.debug_get_field(f)
            out.append(g.cpu())
            del g
        res.append(out)
        ch.close()
    for a, b in zip(*res):
        assert torch.equal(a, b)
