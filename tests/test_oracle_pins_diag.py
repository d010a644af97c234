"""Pins of the oracle's DIAGNOSTIC combinations (no GPU, no CUDA path): the Lagrangian density of PAPER.md:198 Eq. 33
with its scale-factor weights (reading R-14), the velocity-estimator weights of :216-224 Eq. 36-37, the interaction
potential (:224, :260), the Lagrangian length estimator with mu = 2 pi sigma^2 (:270), the bound-state fractions
(:204-208 Eq. 34-35) and the near-branch-cut mask of the winding sweep (reading R-15).

Each pin ties the expression to something other than itself -- the already pinned kicks (variational principle), a
textbook virial theorem, the Euler-Lagrange damping terms of Eq. 13-16, the Bogomolny vortex, hand-built
configurations -- and is chosen so that a flipped sign, a swapped c <-> 1/c or a dropped weight in
oracle.lagrangian / orc_densities / orc_windings fails at least one of them.
"""
import numpy as np
import pytest

import inputs
from oracle import oracle as O
from test_oracle_pins import K0, _uniform_state, line_state, paper_value, vortex_energy


def sum_L(state, dx, K, c):
    return float(np.sum(O.lagrangian(state, dx, K, c)[0]))


# ------------------------------------------------------------------------------- (i) variational pin, c != 1
@pytest.mark.parametrize("c", [1.7, 0.35])
def test_lagrangian_is_the_action_density_of_the_pinned_kicks(c):
    """With the momenta zeroed, Sum_x L_x is minus the potential-type functional whose gradient the (pinned) kicks
    apply: d Sum L / d Re phi(x) = 2 Re[D-D+ phi - c dV/dphi*] = 2 x the scalar kick's right-hand side (Eq. 17-18), and
    d Sum L / d theta_i(x) = [ -sum_j d-_j F_ij + 2 e^2 c Im(phi* D+_i phi) ] / (c e^2 dx) = RHS of Eq. 20-21 / (c e^2 dx).
    Fails on a wrong sign of grad / mag / pot, on c <-> 1/c, on a missing 1/(2 e^2) or dx power."""
    dx = 0.5
    K = O.Couplings(lambda1=2.0, lambda2=1.6, e1=1.0, e2=0.8, eta1=1.0, eta2=1.1, kappa=0.7)
    s = inputs.random_state((5, 6, 7), 12)
    s[inputs.MOM] = 0.0
    r = s.copy()                                     # right-hand sides from the pinned kicks: Pi+ = 0 + 1 * RHS
    O.kick_scalars(r, dx, K, c, 0.0, 1.0)
    O.kick_gauge(r, dx, K, c, 0.0, 1.0)
    h = 1e-5
    rng = np.random.default_rng(5)
    e0 = {8: K.e1, 9: K.e1, 10: K.e1, 14: K.e2, 15: K.e2, 16: K.e2}
    mom_of = {0: 2, 1: 3, 4: 6, 5: 7, 8: 11, 9: 12, 10: 13, 14: 17, 15: 18, 16: 19}
    for comp in inputs.POS:
        for _ in range(2):
            site = tuple(int(rng.integers(0, n)) for n in s.shape[1:])
            sp, sm = s.copy(), s.copy()
            sp[(comp,) + site] += h
            sm[(comp,) + site] -= h
            dS = (sum_L(sp, dx, K, c) - sum_L(sm, dx, K, c)) / (2 * h)
            rhs = r[(mom_of[comp],) + site]
            want = 2.0 * rhs if comp < 8 else rhs / (c * e0[comp] ** 2 * dx)
            assert abs(want) > 1e-3
            assert abs(dS - want) < 2e-6 * max(1.0, abs(want)), (comp, site, dS, want)


# ------------------------------------------------------------------------------- (iii) virial pins
def _time_average_L(s, dx, K, dtau, nsteps):
    acc = {k: 0.0 for k in ("L", "kin", "grad", "elec", "mag", "pot")}
    for _ in range(nsteps):
        O.step(s, dx, K, 0.0, 0.0, 1.0, dtau)
        lag, d = O.lagrangian(s, dx, K, 1.0)
        acc["L"] += float(np.sum(lag))
        for k in ("kin", "grad", "elec", "mag", "pot"):
            acc[k] += float(np.sum(d[k]))
    return {k: v / nsteps for k, v in acc.items()}


@pytest.mark.parametrize("sym", [+1, -1])
def test_virial_scalar_normal_modes(sym):
    """Small oscillation of the uniform fields about the vacuum (the normal modes of pin P-8, omega^2 = (lambda -+ 2
    kappa) sigma^2): a harmonic oscillator, so over whole periods <kinetic> = <potential> and the time average of
    Sum L = kin - pot vanishes to O(amplitude^3).  A flipped sign of kin (or pot) gives 2 <kin>, a wrong relative
    weight or a wrong sign of the kappa term in pot a finite fraction of it."""
    dtau, eps = 0.01, 1e-3
    w = np.sqrt(2.0 - sym * 2 * 0.9)
    nsteps = int(round(3 * 2 * np.pi / w / dtau))                   # three periods
    s = _uniform_state((2, 2, 2), 1.0 + eps, 1.0 + sym * eps)
    av = _time_average_L(s, 0.5, K0, dtau, nsteps)
    assert av["kin"] > 1e-8 and av["grad"] == 0.0 and av["elec"] == 0.0
    assert abs(av["L"]) < 1e-2 * av["kin"], av
    assert abs(av["kin"] - av["pot"]) < 1e-2 * av["kin"], av


def test_virial_photon_modes():
    """(a) Uniform link theta_x = eps on the vacuum: theta'' = -2 e^2 sigma^2 theta (pin P-8), L = elec - grad, so
    <elec> = <grad>: pins the sign of elec and its 1/(2 e^2) against |D+ phi|^2.  (b) A transverse wave
    theta_y = eps cos(k x): omega^2 = khat^2 + 2 e^2 sigma^2 and <elec> = <mag> + <grad>: pins the sign and the
    1/(2 e^2 dx^4) of the magnetic term."""
    dtau, eps, dx = 0.01, 1e-3, 0.5
    K = O.Couplings(e1=1.1)
    w = np.sqrt(2.0) * 1.1
    s = _uniform_state((2, 2, 2), 1.0, 1.0)
    s[8] = eps
    av = _time_average_L(s, dx, K, dtau, int(round(3 * 2 * np.pi / w / dtau)))
    assert av["elec"] > 1e-8 and av["mag"] == 0.0 and av["kin"] < 1e-4 * av["elec"]
    assert abs(av["L"]) < 1e-2 * av["elec"], av
    assert abs(av["elec"] - av["grad"]) < 1e-2 * av["elec"], av
    n = 8
    s = _uniform_state((1, 1, n), 1.0, 1.0)
    kx = 2 * np.pi / (n * dx)
    s[9, 0, 0, :] = eps * np.cos(kx * dx * np.arange(n))
    w = np.sqrt((2 - 2 * np.cos(kx * dx)) / dx ** 2 + 2 * 1.1 ** 2)
    av = _time_average_L(s, dx, K, dtau, int(round(3 * 2 * np.pi / w / dtau)))
    assert av["mag"] > 0.2 * av["elec"] and av["grad"] > 0.2 * av["elec"]
    assert abs(av["L"]) < 1e-2 * av["elec"], av
    assert abs(av["elec"] - av["mag"] - av["grad"]) < 1e-2 * av["elec"], av


@pytest.mark.parametrize("m,beta", [(0.5, 0.0), (0.5, 1.0), (2 / 3, 0.0), (2 / 3, -0.26), (0.9, 0.3)])
def test_scale_factor_weights_reproduce_the_damping_terms(m, beta):
    """Euler-Lagrange: a^2 L_x is the action density, so the weights w_kin(c), w_elec(c) that oracle.lagrangian puts on
    |phi'|^2 and E^2 fix the friction terms of the equations of motion, d ln(a^2 w)/d tau.  Their ratio must be the
    omega / delta = 1 - beta of Eq. 22 (:147) that the (pinned) kicks use: a weight c instead of 1/c on the electric
    term would give 1 + beta."""
    dx, tau, tn, dtau = 0.5, 3.0, 1.7, 0.1
    only_pi = _uniform_state((2, 2, 2), 1.0, 1.0)
    only_pi[2], only_pi[7] = 0.3, -0.2
    only_E = _uniform_state((2, 2, 2), 1.0, 1.0)
    only_E[11], only_E[19] = 0.4, 0.1

    def log_weights(t):
        a, c, _, _ = O.scalars(t, m, beta, dtau, tn)
        lag, d = O.lagrangian(only_pi, dx, K0, c)
        w_kin = np.sum(lag) / np.sum(d["kin"])
        lag, d = O.lagrangian(only_E, dx, K0, c)
        w_el = np.sum(lag) / np.sum(d["elec"])
        assert w_kin > 0 and w_el > 0                      # both enter the Lagrangian with a plus sign
        return np.log(a * a * w_kin), np.log(a * a * w_el)

    h = 1e-4
    k0, e0 = log_weights(tau * (1 - h))
    k1, e1 = log_weights(tau * (1 + h))
    _, _, delta, omega = O.scalars(tau, m, beta, dtau, tn)
    assert np.isclose((e1 - e0) / (k1 - k0), omega / delta, atol=1e-6)
    assert np.isclose(omega / delta, 1.0 - beta, atol=1e-12)
    # and the kinetic friction itself: d ln(a^2 w_kin)/d ln tau = 2 p = alpha p  <->  delta = (1/2) alpha p dtau / tau
    assert np.isclose((k1 - k0) / (2 * h), 2.0 * delta * tau / dtau, atol=1e-6)


# ------------------------------------------------------------------------------- (ii) Bogomolny pin of xi_L
@pytest.mark.parametrize("sector", [0, 1])
def test_lagrangian_length_estimator_on_the_bogomolny_vortex(sector):
    """Static relaxed vortex-antivortex pair (pin P-4), c = 1: dx^3 Sum L = -H to roundoff, so xi_L = sqrt(-mu V / Sum L)
    with mu = 2 pi sigma^2 must equal the winding estimator xi_W = sqrt(V / L) of the same two strings
    (L = 2 strings x length dx) up to sqrt(mu / mu_lattice), i.e. within half the tension pin's 5 % / 1.5 %."""
    for (n, dx, tol) in ((32, 0.5, 0.025), (64, 0.25, 0.0075)):
        s, K = vortex_energy(n, dx, sector)
        d = O.diagnostics(s, dx, K, 1.0)
        assert np.isclose(dx ** 3 * d["sum_L"], -O.energy(s, dx, K), rtol=1e-12)
        tag = "p" if sector == 0 else "q"
        assert d[f"sumW_{tag}"] == 2 and d["cells_pq"] == 0
        vol = n * n * dx ** 3
        assert np.isclose(d["xi_W"], np.sqrt(vol / (2 * dx)), rtol=1e-12)
        assert abs(d["xi_L"] / d["xi_W"] - 1.0) < tol, (n, d["xi_L"], d["xi_W"])


# ------------------------------------------------------------------------------- (iv) V_int by hand
def test_interaction_potential_on_hand_computed_sites():
    """V_int = kappa0 (|phi|^2 - sigma_p^2)(|psi|^2 - sigma_q^2) and Eq. 4 (:52) on numbers worked
    out by hand; at the core of a (1,1) bound state (phi = psi = 0) V_int = kappa0 sigma_p^2 sigma_q^2 = 0.9 for the
    paper's couplings -- its maximum, just above the 0.855 isosurface of Fig. 2 (:260) -- and 0 in either vacuum."""
    K = O.Couplings(lambda1=2.0, lambda2=1.6, e1=1.0, e2=1.0, eta1=1.0, eta2=1.2, kappa=0.7)
    s = np.zeros((20, 1, 1, 4))
    s[0, 0, 0, 0], s[1, 0, 0, 0] = 0.9, 1.2          # |phi|^2 = 2.25 -> a2 = 1.25
    s[5, 0, 0, 0] = 0.5                              # |psi|^2 = 0.25 -> b2 = 0.25 - 1.44 = -1.19
    s[0, 0, 0, 2], s[4, 0, 0, 2] = 1.0, 0.3          # phi in its vacuum
    s[5, 0, 0, 3] = -1.2                             # psi in its vacuum, phi = 0
    d = O.densities(s, 0.5, K)
    v = d["vint"][0, 0]
    assert np.isclose(v[0], 0.7 * 1.25 * -1.19, rtol=1e-14)
    assert np.isclose(v[1], 0.7 * 1.0 * 1.44, rtol=1e-14)            # phi = psi = 0
    assert v[2] == 0.0 and v[3] == 0.0
    pot = d["pot"][0, 0]
    assert np.isclose(pot[0], 0.5 * 1.25 ** 2 + 0.4 * 1.19 ** 2 - 0.7 * 1.25 * -1.19, rtol=1e-14)
    assert np.isclose(pot[3], 0.5 * 1.0, rtol=1e-14)                 # lambda_p/4 sigma_p^4
    core = O.densities(np.zeros((20, 1, 1, 2)), 0.5, K0)["vint"][0, 0, 0]
    assert core == 0.9 and paper_value("vint_isosurface") < core


def test_velocity_weights_localise_on_bound_states():
    """Eq. 36-37 with W = V_int: only sites where BOTH moduli leave their vacuum contribute.  Two moving lumps, one in
    phi alone and one shared: R_V sees the shared one only, R_L both (weights from the pinned L_x)."""
    K = K0
    s = _uniform_state((1, 1, 8), 1.0, 1.0)
    s[0, 0, 0, 1] = 0.5                               # phi-only lump, moving
    s[2, 0, 0, 1] = 0.4
    s[0, 0, 0, 5], s[4, 0, 0, 5] = 0.6, 0.7           # shared lump, moving slower
    s[2, 0, 0, 5] = 0.1
    d = O.diagnostics(s, 0.5, K, 1.0)
    dens = O.densities(s, 0.5, K)
    v = dens["vint"][0, 0]
    assert v[1] == 0.0 and v[5] > 0 and np.count_nonzero(v) == 1
    want = (0.1 ** 2 * v[5]) / (dens["grad"][0, 0, 5] * v[5])
    assert np.isclose(d["sum_kin_V"] / d["sum_grad_V"], want, rtol=1e-13)
    assert np.isclose(d["v2_pq"], 2 * want / (1 + want), rtol=1e-13)          # Eq. 36
    assert not np.isclose(d["v2_L"], d["v2_pq"], rtol=0.05)


# ------------------------------------------------------------------------------- fractions (Eq. 34-35, :188)
def test_bound_state_fractions_on_hand_built_lines():
    """Two p lines, two q lines, ONE of them coincident: L_pq = 8 cells, and the bound length is subtracted from both
    constituents (:188): L_p = L_q = 16 - 8, so f_total = 8/24 and f_p = 1 (Eq. 34-35)."""
    shape = (8, 8, 8)
    p_lines = [((1.5, 3.5), +1), ((5.5, 3.5), -1)]
    q_lines = [((1.5, 3.5), +1), ((5.5, 6.5), -1)]
    d = O.diagnostics(line_state(shape, p_lines, q_lines), 1.0, K0, 1.0)
    assert d["sumW_p"] == 16 and d["sumW_q"] == 16 and d["cells_pq"] == 8
    assert d["L_pq"] == 8.0 and d["L_p"] == 8.0 and d["L_q"] == 8.0
    assert np.isclose(d["f_total"], 1.0 / 3.0) and d["f_p"] == 1.0
    assert np.isclose(d["xi_pq"], np.sqrt(512 / 8.0)) and np.isclose(d["xi_W"], np.sqrt(512 / 24.0))


# ------------------------------------------------------------------------------- (v) near-branch-cut mask
def _links_touching(shape, x0):
    """Brute force: plaquette (o, z, y, x) is flagged iff one of its four links has the site x0 as an end point."""
    nz, ny, nx = shape
    step = {0: (0, 0, 1), 1: (0, 1, 0), 2: (1, 0, 0)}              # direction -> (dz, dy, dx)
    add = lambda p, d: ((p[0] + d[0]) % nz, (p[1] + d[1]) % ny, (p[2] + d[2]) % nx)
    out = np.zeros((3,) + shape, dtype=np.uint8)
    for o, (i, j) in enumerate(((0, 1), (1, 2), (2, 0))):
        for z in range(nz):
            for y in range(ny):
                for x in range(nx):
                    p = (z, y, x)
                    links = [(p, i), (add(p, step[i]), j), (add(p, step[j]), i), (p, j)]
                    out[o, z, y, x] = any(a == x0 or add(a, step[d]) == x0 for a, d in links)
    return out


@pytest.mark.parametrize("via", ["scalar phase", "link phase", "negative link phase", "negative side"])
def test_near_cut_mask_threshold_and_extent(via):
    """Reading R-15: a plaquette is flagged iff one of its four gauge-invariant link angles chi has pi - |chi| < 1e-5.
    One site (or one link) is set so that chi = +-(pi - 0.5e-5) on known links: exactly the plaquettes containing
    those links are flagged; at pi - 2e-5 nothing is."""
    shape = (4, 5, 6)
    x0 = (1, 2, 3)
    for gap, flagged in ((0.5e-5, True), (2e-5, False)):
        s = _uniform_state(shape, 1.0, 1.0)
        ang = np.pi - gap
        if "link phase" in via:
            s[8][x0] = ang if "negative" in via else -ang           # chi_x(x0) = -theta_x(x0) = +-(pi - gap), phases all 0
            want = np.zeros((3,) + shape, dtype=np.uint8)
            z, y, x = x0
            want[0, z, y, x] = want[0, z, y - 1, x] = 1             # P_xy(x0), P_xy(x0 - y)
            want[2, z, y, x] = want[2, z - 1, y, x] = 1             # P_zx(x0), P_zx(x0 - z)
        else:
            sign = -1.0 if via == "negative side" else 1.0
            s[0][x0], s[1][x0] = np.cos(sign * ang), np.sin(sign * ang)
            want = _links_touching(shape, x0)
        W, near = O.windings(s, 1.0, 0)
        if flagged:
            assert np.array_equal(near, want) and near.sum() == (4 if "link phase" in via else 12)
        else:
            assert not near.any()
        assert not O.windings(s, 1.0, 1)[1].any()                   # the q sector is untouched
        if "link phase" not in via:
            assert not W.any()                                      # a single rotated site is not a string
