"""chan_post_strain_norm_static: the one entry point that allocates nothing (its scratch is a file-scope static device
array inside libchan.so, include/chan.h) against the existing chan_post_strain_norm with caller scratch.

Collected last on purpose (pytest -x must not lose the other tests behind it); passes alone in a
fresh process and after the rest of the suite: it builds and binds its own handles and depends on nothing they left."""
import ctypes as C

import numpy as np
import pytest
import torch

import __graft_entry__ as entry
from paper_1808_06461_b200 import inputs

pytestmark = pytest.mark.gpu


@pytest.fixture(scope="module")
def B():
    if not torch.cuda.is_available():
        pytest.skip("no CUDA device")
    entry.build()
    from paper_1808_06461_b200 import binding
    return binding


def rel(a, b):
    a, b = a.cpu().numpy(), b.cpu().numpy()
    return float(np.linalg.norm((a - b).ravel()) / max(np.linalg.norm(b.ravel()), 1e-300))


def test_static_scratch_entry_point_matches_the_existing_path_twice_in_a_row(B):
    c = inputs.config("mid")
    ch = B.Channel(c["nx"], c["ny"], c["nz"], c["lx"], c["lz"], c["y"], c["re"], c["dt"]).bind("cuda:0")
    v, phi, omy = (t.numpy() for t in inputs.fluctuations(c))
    ch.set_state(v, phi, omy, c["U"], c["W"])
    kxc, kzc = c["cut"]
    assert ch.ny * (2 * kzc + 1) * (kxc + 1) * 16 <= int(ch.lib.chan_post_strain_norm_static_limit()) == 4 << 20
    # two different databases, two calls in a row: the second finds the first call's leftovers in the shared scratch
    dbs = []
    for _ in range(2):
        ch.step()
        dbs.append(ch.filter_store(kxc, kzc).clone())
    assert not torch.equal(dbs[0], dbs[1])
    refs = [ch.post_strain_norm(kxc, kzc, db).clone() for db in dbs]           # existing path, caller scratch
    outs = [torch.full_like(refs[0], float("nan")) for _ in dbs]
    torch.cuda.synchronize()
    free0 = torch.cuda.mem_get_info(0)[0]
    alloc0 = torch.cuda.memory_allocated(0)
    for db, out in zip(dbs, outs):
        ch.post_strain_norm_static(kxc, kzc, db, out)                          # back to back, nothing in between
    torch.cuda.synchronize()
    assert torch.cuda.mem_get_info(0)[0] == free0 and torch.cuda.memory_allocated(0) == alloc0     # allocated nothing
    for n, (out, ref) in enumerate(zip(outs, refs)):
        assert bool(torch.isfinite(torch.view_as_real(out)).all()), n
        assert rel(out, ref) < 1e-12, (n, rel(out, ref))                       # the tolerance of the post-processing parity test
        assert torch.equal(out, ref), n                                        # in fact the same kernel: bit for bit
    # a smaller problem after a larger one (stale data beyond its extent), then the first database again
    small = torch.full((ch.ny, 3, 2), float("nan"), dtype=torch.complex128, device="cuda")
    db_small = ch.filter_store(1, 1)
    ch.post_strain_norm_static(1, 1, db_small, small)
    assert torch.equal(small, ch.post_strain_norm(1, 1, db_small))
    again = torch.empty_like(outs[0])
    ch.post_strain_norm_static(kxc, kzc, dbs[0], again)
    assert torch.equal(again, refs[0])
    # argument checks of the new entry point
    lib, h = ch.lib, ch.h
    assert lib.chan_post_strain_norm_static(h, kxc, kzc, None, again.data_ptr()) == B.EINVAL
    assert lib.chan_post_strain_norm_static(h, c["nx"] // 2, kzc, dbs[0].data_ptr(), again.data_ptr()) == B.EINVAL
    unbound = B.Channel(c["nx"], c["ny"], c["nz"], c["lx"], c["lz"], c["y"], c["re"], c["dt"])
    assert lib.chan_post_strain_norm_static(unbound.h, kxc, kzc, dbs[0].data_ptr(), again.data_ptr()) == B.ESTATE
    unbound.close()
    ch.close()


def test_static_scratch_entry_point_rejects_sizes_beyond_its_limit(B):
    """ny (2 kz + 1)(kx + 1) 16 B > 4 MiB: CHAN_ELIMIT with its own message, and nothing is launched or written."""
    c = inputs.config("mid", nx=256, nz=128, ny=129, mesh=("tanh", 2.0))
    ch = B.Channel(c["nx"], c["ny"], c["nz"], c["lx"], c["lz"], c["y"], c["re"], c["dt"]).bind("cuda:0")
    kxc, kzc = 127, 63
    need = c["ny"] * (2 * kzc + 1) * (kxc + 1) * 16
    assert need > int(ch.lib.chan_post_strain_norm_static_limit())
    db = torch.zeros((10, c["ny"], 2 * kzc + 1, kxc + 1), dtype=torch.complex128, device="cuda")
    out = torch.full((c["ny"], 2 * kzc + 1, kxc + 1), 7.0, dtype=torch.complex128, device="cuda")
    n0 = ch.debug_launch_count()
    rc = ch.lib.chan_post_strain_norm_static(ch.h, kxc, kzc, db.data_ptr(), out.data_ptr())
    assert rc == B.ELIMIT == -5
    assert b"static scratch limit" in ch.lib.chan_strerror(rc)
    torch.cuda.synchronize()
    assert ch.debug_launch_count() == n0 and bool((out == 7.0).all())
    with pytest.raises(B.ChanError) as e:
        ch.post_strain_norm_static(kxc, kzc, db, out)
    assert e.value.status == B.ELIMIT
    # just inside the limit on the same handle: 129 x 63 x 32 x 16 B = 4.16 MB <= 4 MiB
    kxc, kzc = 31, 31
    assert c["ny"] * (2 * kzc + 1) * (kxc + 1) * 16 <= int(ch.lib.chan_post_strain_norm_static_limit())
    g = torch.Generator(device="cuda").manual_seed(3)
    db = torch.view_as_complex(torch.randn((10, c["ny"], 2 * kzc + 1, kxc + 1, 2), generator=g, dtype=torch.float64, device="cuda"))
    out = torch.empty((c["ny"], 2 * kzc + 1, kxc + 1), dtype=torch.complex128, device="cuda")
    ch.post_strain_norm_static(kxc, kzc, db, out)
    assert torch.equal(out, ch.post_strain_norm(kxc, kzc, db))
    ch.close()
