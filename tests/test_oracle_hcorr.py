"""Pins of the NEXT-4 variant "Roe solver with H-correction" (PAPER.md:177 names the Roe solver and no
entropy fix; reading R19 in DESIGN.md): eta of a face = half the largest jump of the fast characteristic speeds v_n -+ c_f between
its L and R states; eta^H = the largest eta among the face and the eight transverse faces of its two cells; every wave speed of
the Roe dissipation is raised to max(|lambda_k|, eta^H).

What fixes it without the oracle's own formula: the stationary EXPANSION shock (the textbook failure of the plain Roe flux: it
returns F_L = F_R and keeps the entropy-violating jump for ever) gets the closed-form flux F_L - eta/2 (U_R - U_L) and dissolves;
eta >= max|lambda| turns the flux into the local Lax-Friedrichs flux; eta = 0 is the plain solver bit for bit; and the whole step
keeps the pins of the scheme (uniform state, conservation, div B, symmetry, second order) and needs exactly one more ghost cell.
"""
import numpy as np
import pytest

from paper_1804_03479_b200 import inputs
import harness as H
import waves

GAM = 1.4


def _expansion_shock():
    """Rankine-Hugoniot pair of a stationary Mach-2 shock (gamma = 1.4, textbook relations typed here), ordered so that the flow
    goes from the subsonic to the supersonic side: an entropy-violating stationary jump.  Generic states (rho, vn, vt1, vt2, P, Bt1, Bt2)."""
    M, g = 2.0, GAM
    r1, p1 = 1.0, 1.0
    a1 = np.sqrt(g * p1 / r1)
    u1 = M * a1
    r2 = r1 * (g + 1) * M * M / ((g - 1) * M * M + 2)
    p2 = p1 * (1 + 2 * g / (g + 1) * (M * M - 1))
    u2 = u1 * r1 / r2
    L = np.array([r2, u2, 0.0, 0.0, p2, 0.0, 0.0])        # subsonic side on the left
    R = np.array([r1, u1, 0.0, 0.0, p1, 0.0, 0.0])        # supersonic side on the right: the characteristics u - a diverge
    return L, R


def test_plain_roe_keeps_a_stationary_expansion_shock_and_the_h_correction_does_not(oracle):
    L, R = _expansion_shock()
    FL, FR = oracle.physflux(L, 0.0, GAM), oracle.physflux(R, 0.0, GAM)
    assert np.abs(FL - FR).max() < 1e-14                  # Rankine-Hugoniot with zero speed
    F0, fb = oracle.riemann(2, L, R, 0.0, GAM)
    assert fb == 0 and np.abs(F0 - FL).max() < 1e-13      # the failure: no dissipation on the wave that carries the whole jump
    aL, aR = np.sqrt(GAM * L[4] / L[0]), np.sqrt(GAM * R[4] / R[0])
    eta = 0.5 * ((R[1] - aR) - (L[1] - aL))               # diverging u - a characteristics; the u + a jump is smaller
    assert eta > 0.9 and abs(0.5 * abs((R[1] + aR) - (L[1] + aL))) < eta
    assert abs(oracle.eta_face(L, R, 0.0, GAM) - eta) < 1e-14
    UL, UR = oracle.prim2cons(L, 0.0, GAM), oracle.prim2cons(R, 0.0, GAM)
    # the jump lies on the single wave with lambda = 0 (u - a of the Roe average), whose speed becomes eta; every other wave is faster
    lam = oracle.eig_roe(L, R, 0.0, GAM)[1]
    assert abs(lam[0]) < 1e-12 and np.all(np.abs(lam[3:]) > eta)      # -f is the sonic wave; entropy, +f (and the degenerate ones at v) are faster
    F1, fb = oracle.roe_eta(L, R, 0.0, eta, GAM)
    assert fb == 0 and np.abs(F1 - (FL - 0.5 * eta * (UR - UL))).max() < 1e-12


def test_h_correction_limits(oracle):
    rng = np.random.default_rng(19)
    for _ in range(50):
        WL = np.array([rng.uniform(0.5, 2), *rng.normal(0, 0.5, 3), rng.uniform(0.5, 2), *rng.normal(0, 0.7, 2)])
        WR = WL * (1 + 0.1 * rng.normal(size=7)); WR[0] = abs(WR[0]); WR[4] = abs(WR[4])
        bn = rng.normal()
        F0, fb0 = oracle.riemann(2, WL, WR, bn)
        rc, lam, Rm, Lm, avg = oracle.eig_roe(WL, WR, bn)
        if fb0 or rc:
            continue
        # eta = 0: the plain solver, bit for bit
        assert np.array_equal(oracle.roe_eta(WL, WR, bn, 0.0)[0], F0)
        if lam[0] < 0 < lam[6]:
            # eta below every |lambda_k|: nothing changes
            small = 0.5 * np.abs(lam).min()
            assert np.array_equal(oracle.roe_eta(WL, WR, bn, small)[0], F0)
            # eta above every |lambda_k|: sum_k a_k R_k = U_R - U_L, so the flux is the local Lax-Friedrichs flux with speed eta
            big = 1.5 * np.abs(lam).max()
            FL, FR = oracle.physflux(WL, bn), oracle.physflux(WR, bn)
            UL, UR = oracle.prim2cons(WL, bn), oracle.prim2cons(WR, bn)
            assert np.abs(oracle.roe_eta(WL, WR, bn, big)[0] - (0.5 * (FL + FR) - 0.5 * big * (UR - UL))).max() < 1e-12
    # eta of a face: symmetric under exchange + reflection, zero for equal states, the u - a / u + a jumps for a pure velocity jump
    W = np.array([1.0, 0.3, 0.1, -0.2, 0.8, 0.5, -0.4])
    assert oracle.eta_face(W, W, 0.7) == 0.0
    W2 = W.copy(); W2[1] += 0.6
    assert abs(oracle.eta_face(W, W2, 0.7) - 0.3) < 1e-15


def _tube_with_expansion_shock(n):
    L, R = _expansion_shock()
    nn, NT = 2 * n, 4
    dh = 1.0 / n
    xc = (np.arange(nn) + 0.5) * dh
    # periodic domain of length 2: expansion shock at x = 0.5; the supersonic state leaves through a compressive stationary
    # shock at x = 1.5 (the same Rankine-Hugoniot pair the right way round), which the schemes hold
    left = (xc < 0.5) | (xc >= 1.5)
    o = np.zeros((NT, NT, nn))
    rho = np.where(left, L[0], R[0]) + o; u = np.where(left, L[1], R[1]) + o; p = np.where(left, L[4], R[4]) + o
    bx = np.zeros((NT, NT, nn + 1)); by = np.zeros((NT, NT + 1, nn)); bz = np.zeros((NT + 1, NT, nn))
    return inputs.conserved(rho, u, o, o, p, bx, by, bz, GAM), bx, by, bz, dh, xc


@pytest.mark.parametrize("name,scheme,recon,g", [("vl_plm", 0, 0, 3), ("ctu_ppm", 1, 1, 4)])
def test_expansion_shock_dissolves_only_with_the_h_correction(oracle, name, scheme, recon, g):
    n = 64
    res = {}
    for hc in (0, 1):
        U, bx, by, bz, dh, xc = _tube_with_expansion_shock(n)
        cfg = oracle.make_config(N=4, g=g + hc, gamma=GAM, scheme=scheme, recon=recon, riemann=2, hcorr=hc)
        adv = lambda Ui, Bi, dt, dh_: oracle.advance(cfg, Ui, Bi, dt, dh_)
        for _ in range(40):
            U, bx, by, bz, out, _ = H.step_grid(adv, U, bx, by, bz, 0.3 * dh / 3.6, dh, 4, g + hc)
        r = U[0][0, 0, :]
        w = np.abs(xc - 0.5) < 0.2
        res[hc] = np.abs(np.diff(r[w])).max()
    jump = _expansion_shock()[0][0] - _expansion_shock()[1][0]
    assert res[0] > 0.95 * jump, res          # plain Roe: the whole entropy-violating jump still sits between two cells
    assert res[1] < 0.5 * jump, res           # H-correction: it has opened into a rarefaction fan


SCHEMES = [("vl_plm", 0, 0, 3), ("ctu_ppm", 1, 1, 4)]


@pytest.mark.parametrize("name,scheme,recon,g", SCHEMES)
def test_whole_step_pins_with_h_correction(oracle, name, scheme, recon, g):
    """P2 uniform state, P3 conservation, P4 div B + shared faces, P9 decomposition bitwise with g+1 ghost cells and not with g"""
    gh = g + 1
    cfg = oracle.make_config(N=16, g=gh, scheme=scheme, recon=recon, riemann=2, hcorr=1)
    adv = lambda Ui, Bi, dt, dh_: oracle.advance(cfg, Ui, Bi, dt, dh_)
    n = 16
    bx = np.full((n, n, n + 1), 0.5); by = np.full((n, n + 1, n), -0.3); bz = np.full((n + 1, n, n), 0.9)
    o = np.ones((n, n, n))
    U = inputs.conserved(1.3 * o, 0.4 * o, -0.7 * o, 0.2 * o, 0.8 * o, bx, by, bz)
    Un, bxn, byn, bzn, out, _ = H.step_grid(adv, U, bx, by, bz, 0.01, 1.0 / n, 16, gh)
    assert np.array_equal(bxn, bx) and np.array_equal(byn, by) and np.array_equal(bzn, bz) and np.abs(Un - U).max() < 1e-14
    n = 32
    U, bx, by, bz, dh = inputs.random_group_grid(n, 77)
    t0 = H.totals(U)
    for _ in range(5):
        U1, bx1, by1, bz1, out, mism = H.step_grid(adv, U, bx, by, bz, 0.2 * dh / 3.0, dh, 16, gh)
        U, bx, by, bz = U1, bx1, by1, bz1
        assert mism == 0.0 and H.rel_divb(bx, by, bz, dh) < 1e-13
    t1 = H.totals(U)
    assert abs(t1[0] - t0[0]) / t0[0] < 1e-13 and abs(t1[4] - t0[4]) / t0[4] < 1e-13
    # decomposition: 32^3 as one group = as 8 groups, bitwise, with g+1 ghost cells; the scheme's own width is rejected, and forced, differs
    U, bx, by, bz, dh = inputs.random_group_grid(n, 5)
    dt = 0.2 * dh
    cfgM = oracle.make_config(N=32, g=gh, scheme=scheme, recon=recon, riemann=2, hcorr=1)
    a = H.step_grid(lambda Ui, Bi, dt_, dh_: oracle.advance(cfgM, Ui, Bi, dt_, dh_), U, bx, by, bz, dt, dh, 32, gh)
    b = H.step_grid(adv, U, bx, by, bz, dt, dh, 16, gh)
    for x, y in zip(a[:4], b[:4]):
        assert np.array_equal(x, y)
    plain = H.step_grid(lambda Ui, Bi, dt_, dh_: oracle.advance(oracle.make_config(N=16, g=gh, scheme=scheme, recon=recon, riemann=2), Ui, Bi, dt_, dh_),
                        U, bx, by, bz, dt, dh, 16, gh)
    assert np.abs(plain[0] - b[0]).max() > 1e-8          # and it is not a no-op on this (transonic, config-2 type) state
    cfgS = oracle.make_config(N=16, g=g, scheme=scheme, recon=recon, riemann=2, hcorr=1)
    Ui, Bi = inputs.pack_groups(U, bx, by, bz, 16, g)
    with pytest.raises(ValueError):
        oracle.advance(cfgS, Ui, Bi, dt, dh)
    outS = oracle.advance(cfgS, Ui, Bi, dt, dh, force_ghost_ok=True)
    Us, bxs = inputs.unpack_groups(outS["U"], outS["B"], n, 16)[:2]
    if scheme == 0:      # VL + PLM has no slack: with its own 3 ghost cells the eta of a transverse face is missing at the rim
        assert (not np.array_equal(np.nan_to_num(Us), a[0])) or (not np.array_equal(np.nan_to_num(bxs), a[1]))
    with pytest.raises(ValueError):                       # H-correction is a property of the Roe solver
        oracle.advance(oracle.make_config(N=16, g=gh, scheme=scheme, recon=recon, riemann=1, hcorr=1), Ui, Bi, dt, dh)


@pytest.mark.parametrize("tf", ["permute", "mirror"])
def test_symmetry_with_h_correction(oracle, tf):
    from test_oracle_pins import _permute, _mirror_x
    f = _permute if tf == "permute" else _mirror_x
    n = 16
    U, bx, by, bz, dh = inputs.random_group_grid(n, 11)
    cfg = oracle.make_config(N=16, g=4, scheme=0, recon=0, riemann=2, hcorr=1)
    adv = lambda Ui, Bi, dt, dh_: oracle.advance(cfg, Ui, Bi, dt, dh_)
    ref = H.step_grid(adv, U, bx, by, bz, 0.25 * dh, dh, 16, 4)[:4]
    got = H.step_grid(adv, *f(U, bx, by, bz), 0.25 * dh, dh, 16, 4)[:4]
    for a, b in zip(got, f(*ref)):
        assert np.abs(a - b).max() / np.abs(b).max() < 1e-13


@pytest.mark.slow
def test_linear_wave_stays_second_order_with_h_correction(oracle):
    errs = []
    for N in (16, 32):
        U, bx, by, bz, dh, spd = waves.axis_wave(N, 0, "fast", NT=4)
        cfg = oracle.make_config(N=4, g=4, scheme=0, recon=0, riemann=2, hcorr=1)
        adv = lambda Ui, Bi, dt, dh_: oracle.advance(cfg, Ui, Bi, dt, dh_)
        errs.append(waves.run_period(adv, lambda *a: 0.3 * a[4] / 2.0, U, bx, by, bz, dh, 1.0 / spd, 4, 4)[0])
    assert np.log2(errs[0] / errs[1]) > 1.5, errs


def test_supersonic_shortcut_is_continuous_with_the_h_correction(oracle):
    """plain Roe returns F_L as soon as the slowest wave moves right (lambda_min >= 0), and the dissipation formula tends to F_L
    there.  With eta > 0 the formula gives F_L only for lambda_min >= eta, so R19 takes the shortcut only there: the flux is a
    continuous function of eta (and of the states) across the switch."""
    WL = np.array([1.0, 0.0, 0.1, -0.2, 0.6, np.sqrt(2.0), 0.5])       # P5 background: c_f = 2 along n with B_n = 1
    WR = WL * np.array([1.02, 1.0, 0.9, 1.1, 0.97, 1.01, 0.98])
    WL[1] = WR[1] = 2.2                                                 # slightly supersonic to the right
    rc, lam, _, _, _ = oracle.eig_roe(WL, WR, 1.0)
    assert rc == 0 and 0.05 < lam[0] < 0.4
    FL = oracle.physflux(WL, 1.0)
    assert np.array_equal(oracle.roe_eta(WL, WR, 1.0, 0.0)[0], FL)
    assert np.array_equal(oracle.roe_eta(WL, WR, 1.0, 0.99 * lam[0])[0], FL)
    just_above = oracle.roe_eta(WL, WR, 1.0, lam[0] * (1 + 1e-9))[0]
    assert 0 < np.abs(just_above - FL).max() < 1e-8
    assert np.abs(oracle.roe_eta(WL, WR, 1.0, 3.0 * lam[0])[0] - FL).max() > 1e-4
