"""Pins of the oracle parts that round 1 left unconstrained ("What's weak" 1):
the helium 2x2 solve (C5), the energy equation (C6: heating shares, which density multiplies
which cooling coefficient), the FIXED_OPACITY step and the magnitude clamp of the donor cap.

Expected values come from the ODE system / hand sums written out HERE and from the rate table
tests/golden/rates_appendixA.txt, never from the oracle.  CPU only.

  P15  consistency: one tiny accepted sub-step equals state + h * RHS, with the RHS of the H/He
       network and of the energy equation written out from the physics (
       SURVEY 8(c) C3-C6) and the golden rates at 1e4 K and 1e5 K
  P16  helium closed forms: HeIII -> HeII -> HeI recombination chain (Bateman solution) and the
       coupled H/He photo-ionisation equilibrium in a held radiation field
  P17  photo-heating alone (T at the floor: every cooling rate underflows): e' - e is the sum of
       the absorbed photons times their own eps_gj, with a distinct eps per (group, absorber)
  P18  FIXED_OPACITY: dt c kappa = 1 halves N and F exactly and books V N / 2 as absorbed
       (implicit step N' = N / (1 + dt c kappa): eqs (6)-(7))
  P19  donor cap (reading S11) on a three-cell chain where the cap IS active: every
       cell value after one forward-Euler stage written out by hand, floor_added == 0
"""
import os

import numpy as np
import pytest

from paper_2404_17630_b200.inputs import configs as cfg
from paper_2404_17630_b200.inputs import mesh as M

GOLD = os.path.join(os.path.dirname(__file__), "golden")
KB = 1.380649e-16


def _golden_rates():
    rows = [l.split() for l in open(os.path.join(GOLD, "rates_appendixA.txt")) if l.strip() and l[0] != "#"]
    r4 = {name: float(v4) for _, name, v4, _ in rows}
    r5 = {name: float(v5) for _, name, _, v5 in rows}
    return {1.0e4: r4, 1.0e5: r5}


def _one_cell(oracle_mod, params):
    return oracle_mod.Oracle(M.cartesian(1, 1.0, periodic=False), params)


def _rhs(r, ct, sig, eps, y, nH, N, xHII, xHeII, xHeIII):
    """Time derivatives of the H/He network, the photon densities and the thermal energy, written
    from the physics: photo-ionisation, collisional ionisation (beta), case-B recombination
    (alpha), photo-heating and the cooling function of SURVEY Appendix A ("each cooling term
    multiplies n_e n_ion")."""
    nHe = y * nH
    nHI, nHII = nH * (1 - xHII), nH * xHII
    nHeI, nHeII, nHeIII = nHe * (1 - xHeII - xHeIII), nHe * xHeII, nHe * xHeIII
    ne = nHII + nHeII + 2 * nHeIII
    nabs = np.array([nHI, nHeI, nHeII])
    rate_gj = ct * N[:, None] * sig * nabs[None, :]          # absorptions per volume and time of group g by species j
    dN = -rate_gj.sum(1)
    gam = rate_gj.sum(0)                                     # photo-ionisations per volume and time: HI, HeI, HeII
    dnHII = gam[0] + r["beta_HI"] * ne * nHI - r["alphaB_HII"] * ne * nHII
    dnHeI = -gam[1] - r["beta_HeI"] * ne * nHeI + r["alphaB_HeII"] * ne * nHeII
    dnHeIII = gam[2] + r["beta_HeII"] * ne * nHeII - r["alphaB_HeIII"] * ne * nHeIII
    heat = (rate_gj * eps).sum()
    cool = ne * (r["rcool_HII"] * nHII + r["rcool_HeII"] * nHeII + r["rcool_HeIII"] * nHeIII
                 + r["cicool_HI"] * nHI + r["cicool_HeI"] * nHeI + r["cicool_HeII"] * nHeII
                 + r["cecool_HI"] * nHI + r["cecool_HeII"] * nHeII
                 + r["brems"] * (nHII + nHeII + 4 * nHeIII))
    rates = [np.abs(dN / np.maximum(N, 1e-300)).max(), abs(dnHII) / nH, abs(dnHeI) / max(nHe, 1e-300),
             abs(dnHeIII) / max(nHe, 1e-300)]
    return dN, dnHII / nH, dnHeI / nHe, dnHeIII / nHe, heat - cool, (heat, cool), max(rates)


# states chosen so that every term of every equation carries >= 10 % of its equation in some probe:
# (T, y_he, xHII, xHeII, xHeIII, photons?)
PROBES = [
    (1.0e4, 0.0789, 0.60, 0.50, 0.20, False),   # recombinations + Ly-alpha cooling
    (1.0e4, 0.0789, 0.60, 0.50, 0.20, True),
    (1.0e4, 5.0, 0.999, 0.05, 0.90, False),     # helium-rich, HeIII recombination and its cooling dominate
    (1.0e4, 5.0, 0.999, 0.90, 0.05, False),     # HeII recombination (alpha_HeII, rcool_HeII) dominates
    (1.0e4, 1.0, 0.30, 0.20, 0.10, True),       # photo-ionisation of all three absorbers
    (1.0e5, 0.0789, 0.50, 0.30, 0.30, False),   # collisional ionisation / excitation of H I
    (1.0e5, 5.0, 0.9999, 0.0005, 0.0001, False),  # collisional ionisation of He I (nHeI large)
    (1.0e5, 5.0, 0.9999, 0.98, 0.01, False),    # collisional ionisation + excitation of He II
    (1.0e5, 1.0, 0.9999, 0.02, 0.97, False),    # HeIII recombination against beta_HeII at 1e5 K, bremsstrahlung 4 n_HeIII
    (1.0e5, 1.0, 0.40, 0.40, 0.40, True),
    (1.0e4, 1.0e-3, 0.9999, 0.30, 0.30, False),  # ionised hydrogen: H II recombination cooling against bremsstrahlung
]


@pytest.mark.parametrize("probe", range(len(PROBES)))
def test_p15_tiny_substep_equals_state_plus_h_rhs(oracle_mod, probe):
    T, y, xHII, xHeII, xHeIII, photons = PROBES[probe]
    r = _golden_rates()[T]
    rs = np.random.RandomState(100 + probe)
    nH, ct = 0.7, 2.5e9
    sig = cfg.SIGMA3 * rs.uniform(0.5, 1.5, (3, 3))
    sig[0, 1:] = 0.0; sig[1, 2] = 0.0                       # thresholds: group 1 sees H I only, group 2 not He II
    eps = rs.uniform(2.0, 40.0, (3, 3)) * cfg.EV            # a distinct heating energy per (group, absorber)
    N = rs.uniform(0.5, 2.0, 3) * (1e-6 if photons else 0.0)
    p = cfg.Params(ngroup=3, ctilde=ct, sigma=sig, eps_heat=eps, chem_mode=cfg.CHEM_HHE_THERMAL, y_he=y)
    o = _one_cell(oracle_mod, p)
    e0 = cfg.eth_from_T(T, nH, xHII, xHeII, xHeIII, y)
    dN, dxHII, dxHeI, dxHeIII, de, (heat, cool), fastest = _rhs(r, ct, sig, eps, y, nH, N, xHII, xHeII, xHeIII)
    h = 1.0e-6 / max(fastest, abs(de) / e0)                  # every relative change ~1e-6: one accepted sub-step
    F = np.outer(N, [0.3 * ct, -0.2 * ct, 0.1 * ct])
    out = o.chem_cell(N, F, xHII, xHeII, xHeIII, e0, nH, h)
    assert out["attempts"] == 1
    tol = 1.0e-3                                             # golden table has 5 digits; scheme is O(h) away
    got = {"xHII": (out["xHII"] - xHII) / h, "xHeI": -((out["xHeII"] - xHeII) + (out["xHeIII"] - xHeIII)) / h,
           "xHeIII": (out["xHeIII"] - xHeIII) / h, "e": (out["eth"] - e0) / h}
    want = {"xHII": dxHII, "xHeI": dxHeI, "xHeIII": dxHeIII, "e": de}
    for k in want:
        # relative to the derivative itself, or to 1e-3 of its largest term where terms cancel
        scale = max(abs(want[k]), 1e-3 * (heat + cool) if k == "e" else 0.0)
        ulp = 2.2e-16 * {"xHII": 1.0, "xHeI": 1.0, "xHeIII": 1.0, "e": e0}[k] / h   # rounding of x' - x (fractions are O(1) sums)
        assert abs(got[k] - want[k]) <= tol * scale + 8 * ulp, (k, got[k], want[k])
    if photons:
        assert np.allclose((out["N"] - N) / h, dN, rtol=tol)
        # N and F are absorbed alike (S16): the reduced flux F / N is unchanged
        assert np.allclose(out["F"] / out["N"][:, None], F / N[:, None], rtol=1e-12)


def test_p15_probes_cover_every_term():
    """Each rate coefficient carries >= 10 % of its equation in at least one probe (else a wrong
    coefficient or density could hide below the tolerance)."""
    G = _golden_rates()
    seen = {}
    for T, y, xHII, xHeII, xHeIII, _ in PROBES:
        r = G[T]
        nH = 0.7; nHe = y * nH
        nHI, nHII = nH * (1 - xHII), nH * xHII
        nHeI, nHeII, nHeIII = nHe * (1 - xHeII - xHeIII), nHe * xHeII, nHe * xHeIII
        eqs = {"H": {"beta_HI": r["beta_HI"] * nHI, "alphaB_HII": r["alphaB_HII"] * nHII},
               "HeI": {"beta_HeI": r["beta_HeI"] * nHeI, "alphaB_HeII": r["alphaB_HeII"] * nHeII},
               "HeIII": {"beta_HeII": r["beta_HeII"] * nHeII, "alphaB_HeIII": r["alphaB_HeIII"] * nHeIII},
               "cool": {"rcool_HII": r["rcool_HII"] * nHII, "rcool_HeII": r["rcool_HeII"] * nHeII,
                        "rcool_HeIII": r["rcool_HeIII"] * nHeIII, "cicool_HI": r["cicool_HI"] * nHI,
                        "cicool_HeI": r["cicool_HeI"] * nHeI, "cicool_HeII+cecool_HeII": (r["cicool_HeII"] + r["cecool_HeII"]) * nHeII,
                        "cecool_HI": r["cecool_HI"] * nHI, "brems": r["brems"] * (nHII + nHeII + 4 * nHeIII)}}
        for terms in eqs.values():
            tot = sum(terms.values())
            for k, v in terms.items():
                seen[k] = max(seen.get(k, 0.0), v / tot)
    weak = {k: v for k, v in seen.items() if v < 0.10}
    assert not weak, weak


def test_p16_helium_recombination_chain_closed_form(oracle_mod):
    # hydrogen held ionised (alpha_B,HII overridden to ~0), trace helium: n_e = n_H to 1e-3, so
    # d xHeIII/dt = -a xHeIII, d xHeII/dt = a xHeIII - b xHeII with a = alpha_HeIII n_e, b = alpha_HeII n_e
    r = _golden_rates()[1.0e4]
    nH, y = 2.0e-2, 1.0e-4
    p = cfg.Params(ngroup=1, ctilde=1.0, sigma=np.array([[6.3e-18, 0, 0]]), chem_mode=cfg.CHEM_H_ISOTHERMAL,
                   T_fixed=1.0e4, alphaB_override=1e-40, y_he=y, f_accept=0.02, f_target=0.01)
    o = _one_cell(oracle_mod, p)
    a, b = r["alphaB_HeIII"] * nH, r["alphaB_HeII"] * nH
    x30, x20 = 0.8, 0.15
    t = 1.5 / a
    out = o.chem_cell([0.0], [[0, 0, 0]], 1.0, x20, x30, 1.0, nH, t)
    x3 = x30 * np.exp(-a * t)
    x2 = x20 * np.exp(-b * t) + x30 * a / (a - b) * (np.exp(-b * t) - np.exp(-a * t))
    assert out["xHeIII"] == pytest.approx(x3, rel=0.02)
    assert out["xHeII"] == pytest.approx(x2, rel=0.02)
    assert out["xHII"] == pytest.approx(1.0, abs=1e-6)
    assert out["attempts"] > 100


def test_p16_coupled_photoionisation_equilibrium(oracle_mod):
    # radiation field of group 2 held fixed (reset every call), optically thin: steady state of
    #   Gamma_HI (1 - xHII) = alpha_HII n_e xHII,   Gamma_HeI (1 - xHeII) = alpha_HeII n_e xHeII,
    #   n_e = n_H (xHII + y xHeII);  no HeII-ionising photons and beta_HeII(1e4 K) ~ 1e-37: xHeIII = 0
    r = _golden_rates()[1.0e4]
    nH, y, ct = 1.0e-3, 0.3, 5.0e6
    sHI, sHeI = 4.7461e-19, 1.0e-18
    p = cfg.Params(ngroup=1, ctilde=ct, sigma=np.array([[sHI, sHeI, 0.0]]), chem_mode=cfg.CHEM_H_ISOTHERMAL,
                   T_fixed=1.0e4, y_he=y)
    o = _one_cell(oracle_mod, p)
    N0 = 1.0e-3
    hD = 0.005                                               # optically thin over a call: N - N' = N hD / (1 + hD)
    gH, gHe = ct * sHI * N0 / (1 + hD), ct * sHeI * N0 / (1 + hD)
    dt = hD / (ct * (sHI * nH + sHeI * y * nH))
    x, x2 = 0.05, 0.05
    for _ in range(8000):
        out = o.chem_cell([N0], [[0, 0, 0]], x, x2, 0.0, 1.0, nH, dt)
        x, x2 = out["xHII"], out["xHeII"]
    # collisional ionisation of H I at 1e4 K (beta_HI = 6.2e-16) is 0.2 % of alpha: kept in the balance
    X, X2 = 0.5, 0.5
    for _ in range(200):
        ne = nH * (X + y * X2)
        X = (gH + r["beta_HI"] * ne) / (gH + r["beta_HI"] * ne + r["alphaB_HII"] * ne)
        X2 = gHe / (gHe + r["alphaB_HeII"] * ne)
    assert 0.2 < X < 0.95 and 0.2 < X2 < 0.99                # a non-trivial balance, not saturation
    assert x == pytest.approx(X, rel=0.01)
    assert x2 == pytest.approx(X2, rel=0.01)
    assert out["xHeIII"] < 1e-12


def test_p17_photoheating_with_cooling_off(oracle_mod):
    # T = 10 K (the floor): exp(-T_ion/T) underflows and the recombination cooling of a neutral gas
    # is ~1e-40 of the heating, so e' - e = sum_g sum_j (absorptions of g by j) * eps_gj.
    rs = np.random.RandomState(5)
    nH, y, ct = 1.0e-2, 0.0789, 3.0e9
    sig = cfg.SIGMA3.copy()
    eps = rs.uniform(2.0, 40.0, (3, 3)) * cfg.EV
    p = cfg.Params(ngroup=3, ctilde=ct, sigma=sig, eps_heat=eps, chem_mode=cfg.CHEM_HHE_THERMAL, y_he=y)
    o = _one_cell(oracle_mod, p)
    xHII, xHeII, xHeIII = 1e-8, 0.4, 1e-8                    # HeII present so that all nine (g, j) pairs absorb
    e0 = cfg.eth_from_T(10.0, nH, xHII, xHeII, xHeIII, y)
    nabs = np.array([nH * (1 - xHII), y * nH * (1 - xHeII - xHeIII), y * nH * xHeII])
    N = np.array([3.0, 2.0, 1.0]) * 1e-3 * e0 / (20 * cfg.EV)  # absorbing all of it would add ~1e-3 e0... times h D
    D = ct * (sig * nabs[None, :]).sum(1)
    h = 0.05 / D.max()
    out = o.chem_cell(N, np.zeros((3, 3)), xHII, xHeII, xHeIII, e0, nH, h)
    assert out["attempts"] == 1
    absorbed = N - N / (1 + h * D)                            # implicit photon update over the sub-step (C3)
    share = sig * nabs[None, :] / (sig * nabs[None, :]).sum(1)[:, None]
    want = (absorbed[:, None] * share * eps).sum()
    assert np.allclose(out["N"], N / (1 + h * D), rtol=1e-14)
    assert out["eth"] - e0 == pytest.approx(want, rel=1e-9)
    # and the ionisations: every absorbed photon ionises its absorber
    ion = (absorbed[:, None] * share).sum(0)
    assert (out["xHII"] - xHII) * nH == pytest.approx(ion[0], rel=1e-6)
    assert (out["xHeIII"] - xHeIII) * y * nH == pytest.approx(ion[2], rel=1e-6)
    # (He I is not checked here: at 10 K the recombination He II -> He I outweighs its photo-ionisation)


def test_p18_fixed_opacity_halves_exactly(oracle_mod):
    mesh = M.cartesian(2, 2.0, periodic=True)                # V = 1
    C = mesh.ncell
    ct, dt = 0.5, 0.25
    kappa = np.full(C, 1.0 / (ct * dt))                      # dt c kappa = 1  ->  N' = N / 2
    kappa[3] = 0.0                                           # one transparent cell
    kappa[5] = 3.0 / (ct * dt)                               # and one with N' = N / 4
    p = cfg.Params(ngroup=2, ctilde=ct, chem_mode=cfg.CHEM_FIXED_OPACITY, kappa=kappa)
    rs = np.random.RandomState(2)
    N = rs.uniform(1, 2, (2, C)); F = rs.uniform(-0.2, 0.2, (2, 3, C))
    o = oracle_mod.Oracle(mesh, p)
    o.set_sources(cfg.Sources(np.zeros(0, dtype=np.int32), np.zeros((2, 0))))
    o.set_state(cfg.State(N, F, np.zeros(C), np.zeros(C), np.zeros(C), np.ones(C), np.ones(C)))
    o.chemistry_only(dt)
    s = o.get_state()
    fac = np.full(C, 0.5); fac[3] = 1.0; fac[5] = 0.25
    assert np.array_equal(s["N"], N * fac)                   # powers of two: exact
    assert np.array_equal(s["F"], F * fac)
    led = o.ledger()
    assert np.allclose(led["absorbed"], (N * (1 - fac)).sum(1), rtol=1e-15)


def _chain3():
    """Three unit cubes in a row along x, every outer face reflective."""
    C = 3
    cen = np.array([[0.5, 1.5, 2.5], [0.5, 0.5, 0.5], [0.5, 0.5, 0.5]])
    L, R, nrm, fc = [], [], [], []
    for i in range(2):                                       # interior faces x = 1, 2
        L.append(i); R.append(i + 1); nrm.append([1, 0, 0]); fc.append([i + 1.0, 0.5, 0.5])
    L.append(0); R.append(M.BC_REFLECT); nrm.append([-1, 0, 0]); fc.append([0.0, 0.5, 0.5])
    L.append(2); R.append(M.BC_REFLECT); nrm.append([1, 0, 0]); fc.append([3.0, 0.5, 0.5])
    for i in range(3):
        for ax in (1, 2):
            for sg in (-1, 1):
                n = [0, 0, 0]; n[ax] = sg
                c = [i + 0.5, 0.5, 0.5]; c[ax] += 0.5 * sg
                L.append(i); R.append(M.BC_REFLECT); nrm.append(n); fc.append(c)
    F = len(L)
    return M.Mesh(C, F, np.array([3.0, 1.0, 1.0]), np.zeros(3, dtype=np.int32), np.ones(C), cen, np.ones(F),
                  np.ascontiguousarray(np.array(nrm, dtype=np.float64).T), np.ascontiguousarray(np.array(fc).T),
                  np.array(L, dtype=np.int32), np.array(R, dtype=np.int32))


def _chi(f):
    return (3 + 4 * f * f) / (5 + 2 * np.sqrt(4 - 3 * f * f))


def test_p19_donor_cap_active_three_cell_hand_sum(oracle_mod):
    # c = 1, dt = 1/4, V = A = dx = 1.  Cell 0 almost empty (N = e = 2^-20, F = 0); cell 1: N = 1,
    # F = (1,0,0); cell 2: N = 2, F = (1,0,0).  One forward-Euler stage, second order.
    # Gradients (central differences; reflective ghosts copy N and mirror F) after the limiter:
    #   cell 0: dN/dx = 0 (extrapolating to the wall would undershoot the minimum e), dF/dx = 0
    #   cell 1: dN/dx = (2 - e)/2 (unlimited), dFx/dx = 0 (the right face would overshoot the maximum 1)
    #   cell 2: dN/dx = 0, dFx/dx = 0 (both would overshoot)
    # Face A = (0|1): U_L = (e, 0), U_R = (1/2 + e/4, 1): f_R > 1 -> chi = 1.
    #   Phi_N = 1/2 (0 + 1) - 1/2 (1/2 + e/4 - e) = 1/4 + 3e/8 > 0: donor is cell 0, which holds only
    #   e V / (dt A) = 4e  ->  the cap clamps Phi_N to 4e (and leaves Phi_F alone).
    #   Phi_Fx = 1/2 (e/3 + 1/2 + e/4) - 1/2 (1 - 0) = -1/4 + 7e/24
    # Face B = (1|2): U_L = (3/2 - e/4, 1), U_R = (2, 1): Phi_N = 1 - 1/2 (1/2 + e/4) = 3/4 - e/8,
    #   Phi_Fx = 1/2 (N_L chi(1/N_L) + 2 chi(1/2))
    # Walls: Phi_N = 0; the wall at x = 3 gives Phi_Fx = 2 chi(1/2) + 1, the one at x = 0 gives -e/3;
    # the y and z walls cancel in pairs.
    e = 2.0 ** -20
    mesh = _chain3()
    p = cfg.Params(ngroup=1, ctilde=1.0, chem_mode=cfg.CHEM_NONE, order=2, heun=0, n_floor=0.0)
    N = np.array([[e, 1.0, 2.0]])
    F = np.zeros((1, 3, 3)); F[0, 0] = [0.0, 1.0, 1.0]
    o = oracle_mod.Oracle(mesh, p)
    o.set_sources(cfg.Sources(np.zeros(0, dtype=np.int32), np.zeros((1, 0))))
    o.set_state(cfg.State(N, F, np.zeros(3), np.zeros(3), np.zeros(3), np.ones(3), np.ones(3)))
    gN, gF = o.gradients()
    assert np.allclose(gN[0, 0], [0.0, (2 - e) / 2, 0.0], atol=1e-15) and np.all(gF == 0.0)
    dt = 0.25
    o.step(dt, 1)
    s, led = o.get_state(), o.ledger()
    NL = 1.5 - e / 4
    chiB, chiH = _chi(1.0 / NL), _chi(0.5)
    phiA_N, phiA_F = 4 * e, -0.25 + 7 * e / 24               # capped: without the cap phiA_N = 1/4 + 3e/8
    phiB_N, phiB_F = 0.75 - e / 8, 0.5 * (NL * chiB + 2 * chiH)
    want_N = np.array([e - dt * phiA_N, 1.0 - dt * (phiB_N - phiA_N), 2.0 + dt * phiB_N])
    want_F = np.array([0.0,                                  # |F| <= c N = 0 in the emptied cell (S12)
                       1.0 - dt * (phiB_F - phiA_F), 1.0 - dt * ((2 * chiH + 1) - phiB_F)])
    assert want_N[0] == 0.0                                  # the donor gives exactly what it holds
    assert np.allclose(s["N"][0], want_N, rtol=0, atol=1e-15)
    assert np.allclose(s["F"][0, 0], want_F, rtol=0, atol=1e-15)
    assert np.all(s["F"][0, 1:] == 0.0)
    assert led["floor_added"][0] == 0.0                      # no floor needed: the cap did its job
    assert s["N"][0].sum() == pytest.approx(3.0 + e, abs=1e-15)
