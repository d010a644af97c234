"""CPU-side checks of the boundary: libu1u1.so builds, loads and exports every symbol that
include/u1u1.h declares; size queries and argument validation work without a GPU."""
import ctypes
import os
import re

import pytest

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


@pytest.fixture(scope="module")
def lib():
    from paper_2208_01525_b200 import build, binding
    build.build()
    return binding.load()


def declared_symbols():
    text = open(os.path.join(ROOT, "include", "u1u1.h")).read()
    text = re.sub(r"/\*.*?\*/", "", text, flags=re.S)
    return sorted(set(re.findall(r"\b(u1u1_[a-z_]+)\s*\(", text)))


def test_every_declared_symbol_is_exported(lib):
    from paper_2208_01525_b200 import binding
    names = declared_symbols()
    assert len(names) >= 18
    for n in names:
        assert hasattr(lib, n), f"{n} declared in include/u1u1.h but not exported"
    assert sorted(binding.SYMBOLS) == names


def test_size_queries(lib):
    assert lib.u1u1_state_bytes(64) == 30 * 64 ** 3 * 4
    assert lib.u1u1_state_bytes(1024) == 30 * 1024 ** 3 * 4          # 128.8 GB: fits 180 GB HBM3e
    assert lib.u1u1_scratch_bytes(64) >= 8 * 64 ** 3
    for bad in (0, 4, 7, 66, 1028, -8):
        assert lib.u1u1_state_bytes(bad) == 0 and lib.u1u1_scratch_bytes(bad) == 0


def test_params_struct_matches_header(lib):
    from paper_2208_01525_b200 import Params
    p = Params()
    assert p.struct_size == ctypes.sizeof(Params) == 104
    assert (p.lambda1, p.e1, p.eta1, p.kappa, p.dtau) == (2.0, 1.0, 1.0, 0.9, 0.1)


def test_create_validates_without_gpu(lib):
    ctx = ctypes.c_void_p()
    assert lib.u1u1_create(ctypes.byref(ctx), None, 0, None, 0, None) == -1
    assert b"NULL" in lib.u1u1_last_error(None)
    assert lib.u1u1_create(ctypes.byref(ctx), 0x1001, 10, 0x2000, 10, None) == -1     # misaligned
    # a context over fake (never dereferenced) aligned pointers: host-side validation only
    assert lib.u1u1_create(ctypes.byref(ctx), 0x10000, 30 * 8 ** 3 * 4, 0x20000, 1 << 20, None) == 0
    from paper_2208_01525_b200 import Params
    p = Params()
    assert lib.u1u1_step(ctx, 1, 1.0, 0.5, 1.0) == -4                                  # not configured
    assert lib.u1u1_configure(ctx, 16, 0.5, ctypes.byref(p)) == -2                     # buffers too small
    assert lib.u1u1_configure(ctx, 10, 0.5, ctypes.byref(p)) == -2                     # N % 4
    bad = Params(kappa=1.0)                                                            # kappa >= sqrt(l1 l2)/2
    assert lib.u1u1_configure(ctx, 8, 0.5, ctypes.byref(bad)) == -3
    assert b"kappa" in lib.u1u1_last_error(ctx)
    bad = Params(); bad.struct_size = 8
    assert lib.u1u1_configure(ctx, 8, 0.5, ctypes.byref(bad)) == -1
    assert lib.u1u1_configure(ctx, 8, 0.5, ctypes.byref(p)) == 0
    assert lib.u1u1_step(ctx, 0, 1.0, 0.5, 1.0) == 0                                   # n = 0: no launch
    assert lib.u1u1_step(ctx, 1, 1.0, 1.5, 1.0) == -1                                  # era out of range
    # stability guard: a = tau with s=1 blows up near tau ~ 9.6 (dtau=0.1, dx=0.5), SURVEY 8(c) A-3
    assert lib.u1u1_step(ctx, 1, 12.0, 0.5, 1.0) == -6
    assert b"unstable" in lib.u1u1_last_error(ctx)
    assert lib.u1u1_launch_count(ctx) == 0
    lib.u1u1_destroy(ctx)
