"""u1u1_gauss_violation_static -- the Gauss-law monitor for callers that cannot allocate device memory.

Who needs it: code that lives inside an application whose own memory pool already holds the whole GPU (the 1024^3 run
fills 170 of 178 GiB), or that is called where a cudaMalloc / cudaFree would stall every stream of the device, or that
holds nothing but a checkpoint in the canonical layout.  Such a caller cannot give u1u1_create its scratch buffer, so
this one call reduces through a fixed 256 KiB array inside libu1u1.so and needs no context at all.

What is checked: its eight numbers equal those of the existing path (import the same state into a Lattice, call
u1u1_gauss_violation) within the rtol = 1e-10 that tests/test_gpu_diag.py uses for this state -- on two calls in a
row with DIFFERENT inputs, because the array is shared and keeps the first call's partial sums; then once more with
the first input, on a smaller lattice, whose fewer rows sit underneath the stale ones.  The limit (N <= 1024) and the
other argument checks need no GPU and run in the CPU suite.

This file is named test_zz_* so that pytest collects it last: `-x` stops at the first failure, and a failure here
should not hide the parity tests.  It passes alone in a fresh process (the first call then does the per-device
set-up) and after the rest of the suite."""
import ctypes

import numpy as np
import pytest

import inputs

DX = 0.5


def existing_path(state64, e1, e2, tau, tau_norm):
    """The reference for this test: the context-based monitor on the same fp32 numbers (radiation era, s = 1:
    cG = c = (tau / tau_norm)^2)."""
    import torch
    from paper_2208_01525_b200 import Lattice, Params
    N = state64.shape[1]
    lat = Lattice(N)
    lat.configure(DX, Params(e1=e1, e2=e2, tau_norm=tau_norm))
    lat.import_state(torch.from_numpy(state64.astype(np.float32)))
    lat.set_time(tau, 0.5, 1.0)
    g = lat.gauss_violation()
    lat.close()
    return g


@pytest.mark.gpu
def test_static_scratch_monitor_matches_context_monitor_twice_in_a_row():
    import torch
    from paper_2208_01525_b200 import gauss_violation_static
    dev = torch.device("cuda:0")
    cases = [  # (N, seed, e1, e2, tau, tau_norm)
        (40, 21, 1.1, 0.7, 3.0, 2.0),      # 160 partial rows
        (40, 22, 0.9, 1.3, 2.0, 1.0),      # same rows, other numbers: a stale row would show
        (24, 21, 1.1, 0.7, 3.0, 2.0),      # 96 rows; rows 96..159 still hold the previous call's sums
    ]
    states = [inputs.to_f32_exact(inputs.random_state((N, N, N), seed=seed)) for N, seed, *_ in cases]
    dev_states = [torch.from_numpy(s.astype(np.float32)).to(dev) for s in states]
    outs = [torch.full((8,), float("nan"), dtype=torch.float64, device=dev) for _ in cases]
    # back to back on one stream, no synchronisation in between: the caller's buffers only
    for (N, seed, e1, e2, tau, tau_norm), t, o in zip(cases, dev_states, outs):
        got = gauss_violation_static(t, DX, e1, e2, (tau / tau_norm) ** 2, out=o)
        assert got is o
    torch.cuda.synchronize(dev)
    for (N, seed, e1, e2, tau, tau_norm), s, o in zip(cases, states, outs):
        ref = existing_path(s, e1, e2, tau, tau_norm)
        got = o.cpu().numpy()
        assert np.all(np.isfinite(got)) and np.all(got[[0, 1, 4, 5]] > 0)
        assert np.allclose(got, ref, rtol=1e-10, atol=0), (N, seed, got, ref)
    # and the same call again gives the same bits (fixed reduction order, no atomics)
    again = gauss_violation_static(dev_states[2], DX, cases[2][2], cases[2][3], (cases[2][4] / cases[2][5]) ** 2)
    torch.cuda.synchronize(dev)
    assert np.array_equal(again.cpu().numpy(), outs[2].cpu().numpy())


def test_static_scratch_monitor_rejects_what_it_cannot_do():
    """No GPU needed: the argument checks come before any CUDA call."""
    from paper_2208_01525_b200 import binding, build
    build.build()
    lib = binding.load()
    err = ctypes.create_string_buffer(256)
    call = lambda N, state=0x10000, out=0x20000, dx=0.5: lib.u1u1_gauss_violation_static(
        state, N, dx, 1.0, 1.0, 1.0, out, None, err, len(err))
    assert binding.STATIC_MAX_N == 1024
    assert call(1028) == -2 and b"U1U1_STATIC_MAX_N = 1024" in err.value and b"1028" in err.value
    assert call(4096) == -2
    assert call(10) == -2 and b"multiple of 4" in err.value
    assert call(32, state=None) == -1 and b"NULL" in err.value
    assert call(32, out=None) == -1
    assert call(32, dx=0.0) == -3
    assert call(32, out=0x20004) == -1 and b"aligned" in err.value
    # the message buffer is optional
    assert lib.u1u1_gauss_violation_static(0x10000, 2048, 0.5, 1.0, 1.0, 1.0, 0x20000, None, None, 0) == -2
