"""No-GPU checks of the C-ABI library: it loads, exports every symbol of include/chan.h, validates its
arguments, and its host-computed compact tables agree with the oracle's exact-rational ones."""
import ctypes as C
import os
import re

import numpy as np
import pytest

import __graft_entry__ as entry
from oracle import compact_fd as cfd
from paper_1808_06461_b200 import binding, inputs

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


@pytest.fixture(scope="module")
def lib():
    entry.build()
    return binding.load()


def test_every_declared_symbol_is_exported(lib):
    header = open(os.path.join(ROOT, "include", "chan.h")).read()
    declared = set(re.findall(r"\b(chan_[a-z_]+)\s*\(", header))
    assert declared == set(binding.EXPORTS)
    for name in declared:
        assert hasattr(lib, name), name


def test_argument_validation_without_gpu(lib):
    y = inputs.mesh_cosine(33, 0.7)
    h = C.c_void_p()
    box = binding.Box(2 * np.pi, np.pi, y.ctypes.data_as(C.POINTER(C.c_double)))

    def create(nx, ny, nz, re=180.0, dt=1e-3):
        g = binding.Grid(nx, ny, nz)
        return lib.chan_create(C.byref(h), C.byref(g), C.byref(box), re, dt, None)

    assert create(33, 33, 32) == binding.EINVAL          # odd nx
    assert create(28, 33, 32) == binding.EINVAL          # 3*28/2 = 42 has a factor 7
    assert create(24, 33, 32) == binding.EINVAL          # 3*24/2 = 36 is not a multiple of 8 (include/chan.h)
    assert create(32, 7, 32) == binding.EINVAL           # fewer than 8 mesh points
    assert create(32, 33, 32, re=-1.0) == binding.EINVAL
    yb = y.copy(); yb[5] = yb[4]
    boxb = binding.Box(2 * np.pi, np.pi, yb.ctypes.data_as(C.POINTER(C.c_double)))
    g = binding.Grid(32, 33, 32)
    assert lib.chan_create(C.byref(h), C.byref(g), C.byref(boxb), 180.0, 1e-3, None) == binding.EINVAL
    assert create(32, 33, 32) == binding.OK
    assert lib.chan_workspace_bytes(h) > 12 * 32 * 16 * 33 * 16
    assert lib.chan_substep(h) == binding.ESTATE         # not bound
    assert lib.chan_step(h) == binding.ESTATE
    assert lib.chan_bind(h, None, 0, None) == binding.EINVAL
    assert lib.chan_strerror(binding.ESTATE) == b"call out of order"
    assert lib.chan_destroy(h) == binding.OK


@pytest.mark.parametrize("name", ["cfg1", "cfg2", "mid"])
def test_band_tables_match_the_exact_rational_oracle_tables(lib, name):
    """The library builds its rows in long double with a Chebyshev moment basis; the oracle in exact
    rationals.  They must agree to rounding (reading R5)."""
    c = inputs.config(name)
    ch = binding.Channel(c["nx"], c["ny"], c["nz"], c["lx"], c["lz"], c["y"], c["re"], c["dt"])
    T = ch.debug_band_tables()
    for got, ref in zip(T, cfd.build_operators(c["y"])):
        scale = np.maximum(np.abs(ref).max(axis=1, keepdims=True), 1e-300)  # A2/B2 wall rows are all zero
        assert (np.abs(got - ref) / scale).max() < 2e-15
    ch.close()


def test_tuning_overrides_go_through_the_handle_not_the_environment(lib, monkeypatch):
    """chan.h: "The library reads no environment variable and keeps no global state"."""
    c = inputs.config("mid")
    monkeypatch.setenv("CHAN_TZ", "1")            # the round-1 override: must be ignored now
    monkeypatch.setenv("CHAN_CHUNK_MB", "1")
    ch = binding.Channel(c["nx"], c["ny"], c["nz"], c["lx"], c["lz"], c["y"], c["re"], c["dt"])
    t0 = ch.debug_get_tuning()
    assert t0["tz"] > 1 and t0["chunk_mb"] == 3072 and t0["planes_per_chunk"] == c["ny"] and t0["plane_overlap"] in (1, 2)
    need0 = ch.workspace_bytes()
    ch.debug_set_tuning(tz=2, zthreads=128, chunk_mb=1, xfuse=4)
    t1 = ch.debug_get_tuning()
    assert (t1["tz"], t1["zthreads"], t1["chunk_mb"], t1["xfuse"]) == (2, 128, 1, 4)
    assert 1 <= t1["planes_per_chunk"] < c["ny"] and ch.workspace_bytes() < need0
    for bad in (dict(tz=3), dict(xfuse=5), dict(maxradix_z=13), dict(zthreads=16), dict(plane_overlap=3)):
        with pytest.raises(binding.ChanError) as e:
            ch.debug_set_tuning(**bad)
        assert e.value.status == binding.EINVAL
        assert ch.debug_get_tuning() == t1        # a refused override leaves the handle unchanged
    ch.debug_set_tuning()                         # all zeros: back to the plan's own choice
    assert ch.debug_get_tuning() == t0 and ch.workspace_bytes() == need0
    ch.close()
