"""Pins of the oracle on the paper's 1-D Riemann problems (Table 1).  The exact
regular solutions the paper plots (Torrilhon 2002) are not in this container, so the pins are what any correct
shock-capturing scheme must give without them: the flow stays one-dimensional and B_n constant to the last bit, the
tube is the same along every axis, and the two fast shocks of RJ2a satisfy the Rankine-Hugoniot conditions of Eq. 7
 with ONE speed for all seven components -- a non-conservative update or a wrong flux component
breaks that at first order in the jump."""
import numpy as np
import pytest

from paper_1804_03479_b200 import inputs
import tubes

G = 5.0 / 3.0


def mk(oracle, scheme, recon, g, riemann):
    cfg = oracle.make_config(N=tubes.NT, g=g, scheme=scheme, recon=recon, riemann=riemann)
    adv = lambda Ui, Bi, dt, dh: oracle.advance(cfg, Ui, Bi, dt, dh)
    c0 = oracle.make_config(N=tubes.NT, g=3)

    def dt_fn(U, bx, by, bz, dh):
        Ui, Bi = inputs.pack_groups(U, bx, by, bz, tubes.NT, 0)
        return oracle.dt_reduce(c0, Ui, Bi, 0, dh, 0.3)[0]
    return adv, dt_fn


def flux_eq7(u, Bn):
    """Eq. 7 for the 1-D state (rho, Mn, Mt1, Mt2, e, Bt1, Bt2)"""
    rho, mn, m1, m2, e, b1, b2 = u
    vn, v1, v2 = mn / rho, m1 / rho, m2 / rho
    b2sum = Bn * Bn + b1 * b1 + b2 * b2
    p = (G - 1.0) * (e - 0.5 * rho * (vn * vn + v1 * v1 + v2 * v2) - 0.5 * b2sum)
    pt = p + 0.5 * b2sum
    vb = vn * Bn + v1 * b1 + v2 * b2
    return np.array([rho * vn, rho * vn * vn + pt - Bn * Bn, rho * vn * v1 - Bn * b1, rho * vn * v2 - Bn * b2, (e + pt) * vn - Bn * vb,
                     b1 * vn - Bn * v1, b2 * vn - Bn * v2])


def fast_shocks(P, pr):
    """(speed, largest relative Rankine-Hugoniot residual) of the left- and right-going fast shocks: the outermost jumps
    of the fan; the state behind each is averaged over the plateau between it and the rotational discontinuity"""
    n = P.shape[1]
    rho, out = P[0], []
    iL = next(i for i in range(int(0.15 * n), n) if abs(rho[i] - pr["L"][0]) > 1e-2 * pr["L"][0])
    iR = next(i for i in range(int(0.93 * n), 0, -1) if abs(rho[i] - pr["R"][0]) > 1e-2 * pr["R"][0])
    for far, star in ((P[:, iL - 6], P[:, iL + 4:iL + 22].mean(axis=1)), (P[:, iR + 6], P[:, iR - 21:iR - 3].mean(axis=1))):
        dU, dF = star - far, flux_eq7(star, pr["Bn"]) - flux_eq7(far, pr["Bn"])
        s = dF[0] / dU[0]
        out.append((s, float(np.max(np.abs(dF - s * dU) / (np.abs(dF) + np.abs(s * dU))))))
    return out


@pytest.mark.parametrize("name,scheme,recon,g,riemann,tol", [("vl_plm_hlld", 0, 0, 3, 1, 2e-2), ("ctu_plm_hlld", 1, 0, 3, 1, 2e-3)])
def test_rj2a_fast_shocks_satisfy_rankine_hugoniot(oracle, name, scheme, recon, g, riemann, tol):
    n = 128
    adv, dt_fn = mk(oracle, scheme, recon, g, riemann)
    grid, dh, dts = tubes.run_tube(adv, dt_fn, "rj2a", n, g=g)
    pr = inputs.RIEMANN_PROBLEMS["rj2a"]
    # the undisturbed states are still there at both ends of the analysed part, to the last bit of rho
    P = tubes.profile(grid, n)
    assert abs(P[0, int(0.2 * n)] - pr["L"][0]) < 1e-12 and abs(P[0, n - 1] - pr["R"][0]) < 1e-6
    (sl, rl), (sr, rr) = fast_shocks(P, pr)
    assert rl < tol and rr < tol, (rl, rr)
    # both schemes find the same shocks (measured: -0.958 .. -0.962 and 2.263 .. 2.264); the left one is a shock moving
    # to the left in the lab frame although the gas flows to the right at 1.2
    assert -0.975 < sl < -0.945 and 2.25 < sr < 2.275, (sl, sr)
    # compression by both shocks, and the seven-wave fan keeps density and pressure positive without any floor
    assert P[0].min() > 0.9 and P[0].max() < 1.75


@pytest.mark.parametrize("name", ["rj2a", "torrilhon"])
def test_tube_stays_one_dimensional_and_is_the_same_along_every_axis(oracle, name):
    n = 32
    adv, dt_fn = mk(oracle, 1, 1, 4, 2)                  # the paper's combination: CTU + PPM + Roe
    prof = []
    for axis in range(3):
        grid, dh, dts = tubes.run_tube(adv, dt_fn, name, n, axis=axis, max_steps=12, g=4)
        U, bx, by, bz = grid
        sl = [slice(0, 1)] * 3; sl[2 - axis] = slice(None)
        assert np.array_equal(U, np.broadcast_to(U[(slice(None),) + tuple(sl)], U.shape))      # no transverse structure
        bn = (bx, by, bz)[axis]
        assert np.array_equal(bn, np.full_like(bn, inputs.RIEMANN_PROBLEMS[name]["Bn"]))        # Eq. 13 in 1-D: B_n is constant
        prof.append(tubes.profile(grid, 2 * n, axis))
    assert np.abs(prof[1] - prof[0]).max() < 1e-13 and np.abs(prof[2] - prof[0]).max() < 1e-13
    assert np.abs(prof[0][0] - inputs.RIEMANN_PROBLEMS[name]["L"][0]).max() > 0.05             # and something did happen
