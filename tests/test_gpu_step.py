"""GPU parity of the fused leapfrog step (through the C ABI) against the fp64 oracle, element by element
on identical (fp32-representable) seeded inputs.  Tolerances are north_star's: max relative error per
field group (max|gpu-oracle| / max|oracle|, reading R-16) 1e-5 after 1 step, 1e-3 after 32."""
import os

import numpy as np
import pytest

import inputs
from oracle import oracle as O

pytestmark = pytest.mark.gpu

DX, DTAU = 0.5, 0.1
VARIANTS = [0, 1, 2, 4, 5, 6, 7]  # 0 tiled fp32 difference form (default); 1 reference; 2 tiled plain fp32; 4 tiled fp64 chain; 5/6/7 = 2/4/0 with libm sincosf


def _torch():
    import torch
    return torch


def group_errors(gpu, ref):
    out = {}
    for name, comps in inputs.GROUPS.items():
        den = np.max(np.abs(ref[comps]))
        num = np.max(np.abs(gpu[comps] - ref[comps]))
        out[name] = num / den if den > 0 else num
    return out


def run_gpu(state64, N, params, calls):
    """calls = [(n, tau, m, s), ...]; returns canonical float64 numpy state."""
    from paper_2208_01525_b200 import Lattice
    torch = _torch()
    lat = Lattice(N)
    lat.configure(DX, params)
    lat.import_state(torch.from_numpy(state64.astype(np.float32)))
    for (n, tau, m, s) in calls:
        lat.step(n, tau, m, s)
    out = lat.export_state().cpu().numpy().astype(np.float64)
    return out, lat


@pytest.mark.parametrize("variant", VARIANTS)
def test_config1_one_and_32_steps(variant):
    """BASELINE.json config 1: 64^3, radiation, s=1, tau0=1, seeded uniform random phases."""
    from paper_2208_01525_b200 import Params
    N = 64
    s0 = inputs.to_f32_exact(O.init_random_phase(N, seed=1))
    K = O.Couplings()
    prm = Params(kernel_variant=variant)
    ref = s0.copy()
    O.step(ref, DX, K, 1.0, 0.5, 1.0, DTAU, tau_norm=1.0, n=1)
    gpu, _ = run_gpu(s0, N, prm, [(1, 1.0, 0.5, 1.0)])
    err1 = group_errors(gpu, ref)
    assert max(err1.values()) < 1e-5, err1
    O.step(ref, DX, K, 1.0 + DTAU, 0.5, 1.0, DTAU, tau_norm=1.0, n=31)
    gpu, lat = run_gpu(s0, N, prm, [(32, 1.0, 0.5, 1.0)])
    err32 = group_errors(gpu, ref)
    assert max(err32.values()) < 1e-3, err32
    # Gauss law below 1e-5 relative (config 1 is a roundoff case: radiation, s=1; G-notes)
    g = lat.gauss_violation()
    cG = O.gauss_coefficient(1.0 + 31 * DTAU, 0.5, 1.0, DTAU, 1.0)
    g_ref = O.gauss_violation(inputs.to_f32_exact(gpu), DX, K, cG)
    assert g[3] < 1e-5 and g[7] < 1e-5, g
    assert np.allclose(g[[1, 5]], g_ref[[1, 5]], rtol=1e-5)
    # splitting the 32 steps into several calls gives the bit-identical state
    gpu2, _ = run_gpu(s0, N, prm, [(5, 1.0, 0.5, 1.0), (27, 1.0 + 5 * DTAU, 0.5, 1.0)])
    assert np.array_equal(gpu, gpu2)


@pytest.mark.parametrize("variant", VARIANTS)
@pytest.mark.parametrize("N,m,s,f", [(24, 2 / 3, 1.0, 1.0), (40, 0.5, -1.0, 0.5), (8, 0.0, 1.0, 1.0),
                                      (36, 0.9, 0.0, 1.0), (132, 0.5, 0.0, 1.0)])
def test_generic_state_every_term(variant, N, m, s, f):
    """All 20 components non-trivial, unequal couplings, friction, sizes that are not multiples of the
    tile (ragged tails), minimum size 8, flat / radiation / matter / damping eras, s in {1, 0, -1}."""
    from paper_2208_01525_b200 import Params
    K = O.Couplings(lambda1=2.0, lambda2=1.7, e1=1.0, e2=0.9, eta1=1.0, eta2=1.2, kappa=0.8)
    prm = Params(lambda1=2.0, lambda2=1.7, e1=1.0, e2=0.9, eta1=1.0, eta2=1.2, kappa=0.8, tau_norm=1.5,
                 friction=f, kernel_variant=variant)
    s0 = inputs.to_f32_exact(inputs.random_state((N, N, N), seed=N))
    ref = s0.copy()
    nsteps = 1 if N > 100 else 3
    O.step(ref, DX, K, 2.0, m, s, DTAU, tau_norm=1.5, friction=f, n=nsteps)
    gpu, _ = run_gpu(s0, N, prm, [(nsteps, 2.0, m, s)])
    err = group_errors(gpu, ref)
    assert max(err.values()) < (1e-5 if nsteps == 1 else 3e-5), err


def test_variants_agree_closely():
    """The tiled kernel and the reference kernel evaluate the same formulas in fp32 (different order)."""
    from paper_2208_01525_b200 import Params
    N = 48
    s0 = inputs.to_f32_exact(inputs.random_state((N, N, N), seed=5))
    a, _ = run_gpu(s0, N, Params(kernel_variant=0), [(4, 1.0, 0.5, 1.0)])
    b, _ = run_gpu(s0, N, Params(kernel_variant=1), [(4, 1.0, 0.5, 1.0)])
    assert max(group_errors(a, b).values()) < 5e-6


def test_sector_symmetry_and_periodic_shift_on_gpu():
    """PAPER.md:79 symmetry and translation covariance (exercises every periodic wrap of the kernel)."""
    from paper_2208_01525_b200 import Params
    N = 32
    s0 = inputs.to_f32_exact(inputs.random_state((N, N, N), seed=9))
    prm = Params()
    a, _ = run_gpu(s0, N, prm, [(3, 1.0, 0.5, 1.0)])
    sw = s0.copy()
    sw[0:4], sw[4:8] = s0[4:8], s0[0:4]
    sw[8:14], sw[14:20] = s0[14:20], s0[8:14]
    b, _ = run_gpu(sw, N, prm, [(3, 1.0, 0.5, 1.0)])
    assert np.array_equal(a[0:4], b[4:8]) and np.array_equal(a[8:14], b[14:20])
    sh = np.roll(s0, shift=(5, -7, 13), axis=(1, 2, 3))
    c, _ = run_gpu(sh, N, prm, [(3, 1.0, 0.5, 1.0)])
    assert np.array_equal(np.roll(a, shift=(5, -7, 13), axis=(1, 2, 3)), c)


def test_error_paths_on_gpu():
    from paper_2208_01525_b200 import Lattice, Params, U1U1Error
    lat = Lattice(16)
    with pytest.raises(U1U1Error, match="ESTATE"):
        lat.step(1, 1.0, 0.5, 1.0)
    lat.init_fields(3, DX, Params())
    with pytest.raises(U1U1Error, match="EUNSTABLE"):
        lat.step(1, 20.0, 0.5, 1.0)
    with pytest.raises(U1U1Error, match="ESTATE"):
        lat.export_windings(0)
    lat.step(2, 1.0, 0.5, 1.0)
    assert lat.launch_count() == 3


@pytest.mark.parametrize("variant", [0, 2, 4, 1])
def test_degenerate_states(variant):
    """All-zero fields stay exactly zero (atan2(0,0)=0, no NaN from the phasors); the uniform vacuum
    |phi|=eta1, |psi|=eta2 with zero links and momenta is an exact fixed point in fp32."""
    from paper_2208_01525_b200 import Lattice, Params
    import torch
    N = 40
    prm = Params(eta2=1.25, kernel_variant=variant)
    for kind in ("zero", "vacuum"):
        s0 = np.zeros((20, N, N, N))
        if kind == "vacuum":
            s0[0], s0[5] = 1.0, -1.25
        lat = Lattice(N)
        lat.configure(DX, prm)
        lat.import_state(torch.from_numpy(s0.astype(np.float32)))
        lat.step(5, 1.0, 0.5, 1.0)
        out = lat.export_state().cpu().numpy().astype(np.float64)
        assert np.array_equal(out, s0), kind
        d = lat.diagnostics()
        assert d["sumW_p"] == 0 and d["sumW_q"] == 0 and d["cells_pq"] == 0 and d["near_p"] == 0
        g = lat.gauss_violation()
        assert g[0] == 0 and g[4] == 0


def test_growth_then_physical_schedule():
    """SURVEY 8(f)-4 / PAPER.md:328-339 Table III: a core-growth phase (beta = beta_growth < 0, a normalised to 1 at
    its start) followed by physical evolution (beta = 1, a normalised to 1 at the end) is a sequence of `step`
    calls with `set_params` in between; here on a short schedule, against the oracle doing the same."""
    from paper_2208_01525_b200 import Lattice, Params
    import torch
    N, n1, n2 = 48, 12, 12
    beta_g = float([l.split()[1] for l in open(os.path.join(os.path.dirname(__file__), "golden", "paper_values.txt"))
                    if l.startswith("table3_beta_growth_rad")][0])
    tau0, tau_tr = 5.0, 5.0 + n1 * DTAU
    tau_end = tau_tr + n2 * DTAU
    s0 = inputs.to_f32_exact(inputs.random_state((N, N, N), seed=77, amp_mom=0.1, amp_theta=0.3))
    K = O.Couplings()
    ref = s0.copy()
    O.step(ref, DX, K, tau0, 0.5, beta_g, DTAU, tau_norm=tau0, n=n1)
    O.step(ref, DX, K, tau_tr, 0.5, 1.0, DTAU, tau_norm=tau_end, n=n2)
    lat = Lattice(N)
    prm = Params(tau_norm=tau0)
    lat.configure(DX, prm)
    lat.import_state(torch.from_numpy(s0.astype(np.float32)))
    lat.step(n1, tau0, 0.5, beta_g)
    prm.tau_norm = tau_end
    lat.set_params(prm)
    lat.step(n2, tau_tr, 0.5, 1.0)
    gpu = lat.export_state().cpu().numpy().astype(np.float64)
    err = group_errors(gpu, ref)
    assert max(err.values()) < 1e-4, err
    d = lat.diagnostics()
    assert np.isclose(d["a"], 1.0) and np.isclose(d["tau"], tau_end)     # width normalised to 1 at the end


@pytest.mark.parametrize("config", [2, 3, 4, 5])
def test_baseline_configs_first_32_steps(config):
    """BASELINE.json configs 2-5 at 64^3 (their own seeds, initial conditions, eras, s, tau_norm and friction
    prephase as scheduled by paper_2208_01525_b200.run_config): the first 32 steps against the oracle from the
    oracle's OWN seeded initial condition (so the generator, the coefficients and the kernel are all in the loop)."""
    from paper_2208_01525_b200 import Lattice, Params
    from paper_2208_01525_b200.run_config import CONFIGS, TAU0
    c = CONFIGS[config]
    N, n = 64, 32
    total = c["pre"] + c["steps"]
    tau_norm = c["tau_norm"] if c["tau_norm"] is not None else TAU0 + total * DTAU
    f = 0.5 if c["pre"] else 1.0
    K = O.Couplings()
    ref = O.init_smoothed(N, config) if c["kind"] == 1 else O.init_random_phase(N, config)
    ref = inputs.to_f32_exact(ref)
    lat = Lattice(N)
    lat.init_fields(config, DX, Params(init_kind=c["kind"], tau_norm=tau_norm, friction=f))
    g0 = lat.export_state().cpu().numpy().astype(np.float64)
    assert np.max(np.abs(g0 - ref)) < 2e-7          # both generators: one fp32 rounding of the fp64 value
    lat.step(n, TAU0, c["m"], c["s"])
    O.step(ref, DX, K, TAU0, c["m"], c["s"], DTAU, tau_norm=tau_norm, friction=f, n=n)
    gpu = lat.export_state().cpu().numpy().astype(np.float64)
    err = group_errors(gpu, ref)
    assert max(err.values()) < 1e-3, err


@pytest.mark.parametrize("base", [0, 2, 4])
def test_staging_paths_bit_identical(base):
    """The tiled kernel stages interior tiles by TMA boxes and boundary tiles by cp.async, momenta by TMA boxes or
    ld.global.cs: the arithmetic is the same, so forcing the other staging path (tuning flags 2 and 4 in bits 4.. of
    kernel_variant) must give the bit-identical state -- on a lattice with interior, boundary and ragged tiles."""
    from paper_2208_01525_b200 import Params
    N = 132
    s0 = inputs.to_f32_exact(inputs.random_state((N, N, N), seed=31))
    outs = []
    for flags in (0, 2, 4):
        out, _ = run_gpu(s0, N, Params(kernel_variant=base + 16 * flags, tau_norm=1.5), [(3, 2.0, 0.5, 1.0)])
        outs.append(out)
    assert np.array_equal(outs[0], outs[1]) and np.array_equal(outs[0], outs[2])


def test_packed_chain_bit_identical_to_scalar_chain():
    """The default kernel runs both sectors through packed fp32x2 instructions (FFMA2 / FADD2 / FMUL2): the same IEEE
    operations in the same order as the scalar difference-form chain (tuning flag 1), so the states must be bit-identical
    -- with unequal couplings in the two sectors, friction, and on interior, boundary and ragged tiles."""
    from paper_2208_01525_b200 import Params
    N = 132
    s0 = inputs.to_f32_exact(inputs.random_state((N, N, N), seed=37))
    outs = []
    for flags in (0, 1, 1 + 2):
        prm = Params(lambda1=2.0, lambda2=1.7, e1=1.0, e2=0.8, eta1=1.0, eta2=1.1, kappa=0.6, friction=0.9,
                     kernel_variant=16 * flags, tau_norm=1.5)
        out, _ = run_gpu(s0, N, prm, [(3, 2.0, 0.5, 1.0), (2, 2.3, 0.5, -1.0)])
        outs.append(out)
    assert np.array_equal(outs[0], outs[1]) and np.array_equal(outs[0], outs[2])


@pytest.mark.parametrize("variant,tol", [(0, 2e-5), (16 * 2048, 1e-5), (7, 1e-5), (4, 2e-5)])
def test_large_link_phases(variant, tol):
    """Non-compact links far outside (-pi, pi] (|theta| up to ~40, reading R-9): the SFU phasor's error grows like
    6e-8 |theta| (documented in step_tiled.cu); with the explicit range reduction of tuning flag 2048 (Cody-Waite,
    f32x2.cuh) the default chain stays at the 1e-5 bar like the libm variants."""
    from paper_2208_01525_b200 import Params
    N = 24
    s0 = inputs.to_f32_exact(inputs.random_state((N, N, N), seed=3, amp_theta=12.0))
    assert np.max(np.abs(s0[[8, 9, 10, 14, 15, 16]])) > 30
    ref = s0.copy()
    O.step(ref, DX, O.Couplings(), 1.0, 0.5, 1.0, DTAU, n=1)
    gpu, _ = run_gpu(s0, N, Params(kernel_variant=variant), [(1, 1.0, 0.5, 1.0)])
    err = group_errors(gpu, ref)
    assert max(err.values()) < tol, err


def test_range_reduce_automatic():
    """u1u1_params.range_reduce = 2: off until a diagnostics sweep reports max |theta| > 10, on from then until the next
    configure.  Before the sweep the step equals range_reduce = 0 bit for bit, after it range_reduce = 1."""
    import torch
    from paper_2208_01525_b200 import Lattice, Params
    N = 24
    s0 = inputs.to_f32_exact(inputs.random_state((N, N, N), seed=3, amp_theta=12.0)).astype(np.float32)

    def one_step(range_reduce, sweep_first):
        lat = Lattice(N)
        lat.configure(DX, Params(range_reduce=range_reduce))
        lat.import_state(torch.from_numpy(s0))
        if sweep_first:
            assert lat.diagnostics()["max_theta"] > 30
        lat.step(1, 1.0, 0.5, 1.0)
        return lat.export_state().cpu().numpy()

    off, on = one_step(0, False), one_step(1, False)
    assert not np.array_equal(off, on)                      # at |theta| ~ 40 the two phasors differ
    assert np.array_equal(one_step(2, False), off)
    assert np.array_equal(one_step(2, True), on)
    assert np.array_equal(one_step(0, True), off)           # the sweep alone changes nothing
