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
    # the experimental switches live in a header of their own, outside the supported boundary
    tuning = re.sub(r"/\*.*?\*/", "", open(os.path.join(ROOT, "include", "u1u1_tuning.h")).read(), flags=re.S)
    tnames = sorted(set(re.findall(r"\b(u1u1_[a-z_]+)\s*\(", tuning)))
    assert tnames == sorted(binding.TUNING_SYMBOLS) and all(hasattr(lib, n) for n in tnames)
    main = open(os.path.join(ROOT, "include", "u1u1.h")).read()
    assert "16*" not in main and "set_tuning" not in main


def test_size_queries(lib):
    assert lib.u1u1_state_bytes(64) == 30 * 64 ** 3 * 4
    assert lib.u1u1_state_bytes(1024) == 30 * 1024 ** 3 * 4          # 128.8 GB: fits 180 GB HBM3e
    assert lib.u1u1_scratch_bytes(64) >= 8 * 64 ** 3
    assert lib.u1u1_aux_bytes(64) == 10 * 64 ** 3 * 4 and lib.u1u1_aux_bytes(66) == 0
    # state + second momentum buffer + scratch at 1024^3 fit the 178.4 GiB a B200 reports
    assert lib.u1u1_state_bytes(1024) + lib.u1u1_aux_bytes(1024) + lib.u1u1_scratch_bytes(1024) < 172 * 2 ** 30
    for bad in (0, 4, 7, 66, 1028, -8):
        assert lib.u1u1_state_bytes(bad) == 0 and lib.u1u1_scratch_bytes(bad) == 0


def test_params_struct_matches_header(lib):
    from paper_2208_01525_b200 import Params
    p = Params()
    assert p.struct_size == ctypes.sizeof(Params) == 112
    assert (p.lambda1, p.e1, p.eta1, p.kappa, p.dtau) == (2.0, 1.0, 1.0, 0.9, 0.1)
    assert (p.kernel_variant, p.range_reduce, p.reserved, p.tuning) == (0, 0, 0, 0)
    # the binding splits the tests' shorthand variant + 16 * switches; the C struct only ever holds 0..7
    q = Params(kernel_variant=4 + 16 * (2 | 512))
    assert (q.kernel_variant, q.tuning, q.range_reduce) == (4, 2 | 512, 0)
    q = Params(kernel_variant=16 * 2048)
    assert (q.kernel_variant, q.tuning, q.range_reduce) == (0, 0, 1)


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
    bad = Params(); bad.kernel_variant = 16                                            # switches are not part of the struct any more
    assert lib.u1u1_configure(ctx, 8, 0.5, ctypes.byref(bad)) == -1
    bad = Params(range_reduce=3)
    assert lib.u1u1_configure(ctx, 8, 0.5, ctypes.byref(bad)) == -1 and b"range_reduce" in lib.u1u1_last_error(ctx)
    assert lib.u1u1_set_tuning(ctx, 4096) == -1 and lib.u1u1_set_tuning(ctx, 2 | 512) == 0 and lib.u1u1_set_tuning(ctx, 0) == 0
    assert lib.u1u1_configure(ctx, 8, 0.5, ctypes.byref(Params(range_reduce=2))) == 0
    assert lib.u1u1_configure(ctx, 8, 0.5, ctypes.byref(p)) == 0
    assert lib.u1u1_step(ctx, 0, 1.0, 0.5, 1.0) == 0                                   # n = 0: no launch
    assert lib.u1u1_step(ctx, 1, 1.0, 1.5, 1.0) == -1                                  # era out of range
    # stability guard: a = tau with s=1 blows up near tau ~ 9.6 (dtau=0.1, dx=0.5), SURVEY 8(c) A-3
    assert lib.u1u1_step(ctx, 1, 12.0, 0.5, 1.0) == -6
    assert b"unstable" in lib.u1u1_last_error(ctx)
    assert lib.u1u1_launch_count(ctx) == 0
    lib.u1u1_destroy(ctx)


C_CLIENT = r"""
/* A plain C99 client of include/u1u1.h: the header must compile as C, and the error paths must work without a GPU. */
#include <stdio.h>
#include <string.h>
#include "u1u1.h"

int main(void)
{
    u1u1_ctx *ctx = NULL;
    u1u1_params p;
    double out[U1U1_DIAG_LEN];
    if (u1u1_state_bytes(64) != (size_t)30 * 64 * 64 * 64 * 4) return 1;
    if (u1u1_scratch_bytes(64) < (size_t)10 * 64 * 64 * 64) return 2;
    if (u1u1_state_bytes(66) != 0) return 3;
    if (u1u1_create(&ctx, NULL, 0, NULL, 0, NULL) != U1U1_EINVAL) return 4;
    if (!strstr(u1u1_last_error(NULL), "NULL")) return 5;
    if (u1u1_create(&ctx, (void *)0x10000, (size_t)30 * 512 * 4, (void *)0x20000, (size_t)1 << 20, NULL) != U1U1_OK) return 6;
    memset(&p, 0, sizeof p);
    p.struct_size = (uint32_t)sizeof p;
    p.lambda1 = p.lambda2 = 2.0; p.e1 = p.e2 = 1.0; p.eta1 = p.eta2 = 1.0; p.kappa = 0.9;
    p.dtau = 0.1; p.tau_norm = 1.0; p.friction = 1.0; p.smooth_width = 5.0; p.smooth_trunc = 20;
    if (u1u1_step(ctx, 1, 1.0, 0.5, 1.0) != U1U1_ESTATE) return 7;
    if (u1u1_aux_bytes(64) != (size_t)10 * 64 * 64 * 64 * 4) return 20;
    if (u1u1_set_aux(NULL, NULL, 0) != U1U1_EINVAL) return 21;
    if (u1u1_set_aux(ctx, (void *)0x30001, (size_t)1 << 20) != U1U1_ESIZE) return 22;      /* misaligned */
    if (u1u1_configure(ctx, 16, 0.5, &p) != U1U1_ESIZE) return 8;
    p.kappa = 1.0;
    if (u1u1_configure(ctx, 8, 0.5, &p) != U1U1_EPARAM) return 9;
    p.kappa = 0.9;
    if (u1u1_configure(ctx, 8, 0.5, &p) != U1U1_OK) return 10;
    if (u1u1_step(ctx, 1, 12.0, 0.5, 1.0) != U1U1_EUNSTABLE) return 11;
    if (u1u1_cool(ctx, 1, 0.05) != U1U1_EUNSTABLE) return 12;
    if (u1u1_export_windings(ctx, 0, NULL, NULL, NULL) != U1U1_ESTATE) return 13;
    if (u1u1_pq_segments(ctx, 1, 0, out) != U1U1_ESTATE) return 14;
    if (u1u1_diagnostics(ctx, NULL) != U1U1_EINVAL) return 15;
    if (u1u1_launch_count(ctx) != 0) return 16;
    printf("%s\n", u1u1_last_error(ctx));
    u1u1_destroy(ctx);
    return U1U1_D_USED <= U1U1_DIAG_LEN ? 0 : 17;
}
"""


def test_header_compiles_as_c99_and_links(lib, tmp_path):
    """include/u1u1.h is a C header: a C99 client built with gcc -std=c99 -Wall -Werror -pedantic links against
    libu1u1.so and exercises the size queries and every error path that needs no GPU."""
    import subprocess
    src = tmp_path / "client.c"
    src.write_text(C_CLIENT)
    exe = tmp_path / "client"
    pkg = os.path.join(ROOT, "paper_2208_01525_b200")
    subprocess.check_call(["gcc", "-std=c99", "-Wall", "-Wextra", "-Werror", "-pedantic", "-I", os.path.join(ROOT, "include"),
                           "-o", str(exe), str(src), "-L", pkg, "-l:libu1u1.so", f"-Wl,-rpath,{pkg}"])
    r = subprocess.run([str(exe)], capture_output=True, text=True)
    assert r.returncode == 0, (r.returncode, r.stdout, r.stderr)
    assert "needs u1u1_diagnostics" in r.stdout or "NULL" in r.stdout


def test_create_error_is_per_thread(lib):
    """The message of a failed u1u1_create lives in thread-local storage: two host threads do not race on it."""
    import threading
    seen = {}

    def worker(tag, misaligned):
        ctx = ctypes.c_void_p()
        if misaligned:
            rc = lib.u1u1_create(ctypes.byref(ctx), 0x1001, 10, 0x2000, 10, None)
        else:
            rc = lib.u1u1_create(ctypes.byref(ctx), None, 0, None, 0, None)
        seen[tag] = (rc, lib.u1u1_last_error(None))

    ts = [threading.Thread(target=worker, args=("a", True)), threading.Thread(target=worker, args=("b", False))]
    for t in ts:
        t.start()
    for t in ts:
        t.join()
    assert seen["a"][0] == -1 and b"aligned" in seen["a"][1]
    assert seen["b"][0] == -1 and b"NULL" in seen["b"][1]
