"""Pins of the CFL reduction `mhdref_dt` and of `fastspeed` (PAPER.md:172 "determined by the CFL condition", :250;
reading R13: dt = C dh / max over interior cells and directions of |v_d| + c_f,d) against closed forms typed here.

Background of pin P5: rho = 1, P = 3/5 (gamma = 5/3 => a^2 = 1), B = (1, sqrt 2, 1/2), |B|^2 = 13/4.
The fast speed along n solves c^4 - (a^2 + |B|^2/rho) c^2 + a^2 B_n^2/rho = 0:
  along x (B_n^2 = 1):   c_f^2 = (17/4 + sqrt(289/16 - 4))/2 = (17/4 + 15/4)/2 = 4      => c_f = 2 exactly
  along y (B_n^2 = 2):   c_f^2 = (17/4 + sqrt(289/16 - 8))/2 = (17 + sqrt 161)/8
  along z (B_n^2 = 1/4): c_f^2 = (17/4 + sqrt(289/16 - 1))/2 = (17 + sqrt 273)/8
"""
import numpy as np
import pytest

from paper_1804_03479_b200 import inputs

G = 5.0 / 3.0
CFX, CFY, CFZ = 2.0, np.sqrt((17.0 + np.sqrt(161.0)) / 8.0), np.sqrt((17.0 + np.sqrt(273.0)) / 8.0)


def _uniform_groups(ngroups, N, g, rho, v, P, B):
    T = N + 2 * g
    bx = np.full((T, T, T + 1), B[0]); by = np.full((T, T + 1, T), B[1]); bz = np.full((T + 1, T, T), B[2])
    o = np.ones((T, T, T))
    U = inputs.conserved(rho * o, v[0] * o, v[1] * o, v[2] * o, P * o, bx, by, bz, G)
    Ui = np.tile(U.reshape(1, -1), (ngroups, 1))
    Bi = np.tile(np.concatenate([bx.ravel(), by.ravel(), bz.ravel()])[None], (ngroups, 1))
    return Ui, Bi


def test_fastspeed_closed_forms(oracle):
    # generic 1-D state W = (rho, vn, vt1, vt2, P, Bt1, Bt2), normal field passed separately
    s2 = np.sqrt(2.0)
    assert abs(oracle.fastspeed([1, 0, 0, 0, 0.6, s2, 0.5], 1.0) - CFX) < 1e-15
    assert abs(oracle.fastspeed([1, 0, 0, 0, 0.6, 0.5, 1.0], s2) - CFY) < 1e-15
    assert abs(oracle.fastspeed([1, 0, 0, 0, 0.6, 1.0, s2], 0.5) - CFZ) < 1e-15
    # the velocity does not enter; B = 0 gives the sound speed; perpendicular propagation gives sqrt(a^2 + b^2)
    assert abs(oracle.fastspeed([1, 7.0, -3.0, 2.0, 0.6, s2, 0.5], 1.0) - CFX) < 1e-15
    assert abs(oracle.fastspeed([2.0, 0, 0, 0, 1.2, 0, 0], 0.0, gamma=1.4) - np.sqrt(1.4 * 1.2 / 2.0)) < 1e-15
    assert abs(oracle.fastspeed([2.0, 0, 0, 0, 1.2, 0.6, 0.8], 0.0, gamma=1.4) - np.sqrt((1.4 * 1.2 + 1.0) / 2.0)) < 1e-15
    # parallel propagation (B_t = 0): the larger of the sound and Alfven speeds
    assert abs(oracle.fastspeed([1.0, 0, 0, 0, 0.6, 0, 0], 3.0) - 3.0) < 1e-15
    assert abs(oracle.fastspeed([1.0, 0, 0, 0, 0.6, 0, 0], 0.5) - 1.0) < 1e-15


@pytest.mark.parametrize("ng", [0, 3])
def test_dt_of_the_p5_background(oracle, ng):
    """at rest the largest signal speed is the fast speed of the direction with the SMALLEST normal field: z"""
    N, dh, cfl = 8, 1.0 / 8, 0.3
    Ui, Bi = _uniform_groups(2, N, ng, 1.0, (0.0, 0.0, 0.0), 0.6, (1.0, np.sqrt(2.0), 0.5))
    cfg = oracle.make_config(N=N, g=3)
    dt, smax = oracle.dt_reduce(cfg, Ui, Bi, ng, dh, cfl)
    assert CFZ > CFX > CFY
    assert abs(smax - CFZ) < 1e-15 and abs(dt - cfl * dh / CFZ) < 1e-15 * dt
    # the same state with the axes relabelled cyclically: the maximum moves with the field, dt does not change
    for B in ((0.5, 1.0, np.sqrt(2.0)), (np.sqrt(2.0), 0.5, 1.0)):
        Ur, Br = _uniform_groups(2, N, ng, 1.0, (0.0, 0.0, 0.0), 0.6, B)
        assert abs(oracle.dt_reduce(cfg, Ur, Br, ng, dh, cfl)[1] - CFZ) < 1e-15
    # dt is linear in the CFL number and in dh
    dt2, _ = oracle.dt_reduce(cfg, Ui, Bi, ng, 0.5 * dh, 0.5 * cfl)
    assert abs(dt2 - 0.25 * dt) < 1e-15 * dt


def test_dt_of_a_moving_state_takes_the_largest_direction_and_the_magnitude_of_v(oracle):
    N, ng, dh, cfl = 8, 3, 0.01, 0.5
    v = (0.3, -2.5, 0.1)                       # |v_y| + c_f,y is the largest: a signed v or a sum over directions would differ
    Ui, Bi = _uniform_groups(1, N, ng, 1.0, v, 0.6, (1.0, np.sqrt(2.0), 0.5))
    cfg = oracle.make_config(N=N, g=3)
    dt, smax = oracle.dt_reduce(cfg, Ui, Bi, ng, dh, cfl)
    expect = max(0.3 + CFX, 2.5 + CFY, 0.1 + CFZ)
    assert expect == 2.5 + CFY
    assert abs(smax - expect) < 4e-15 and abs(dt - cfl * dh / expect) < 4e-15 * dt
    # density scaling: rho -> 4 rho at fixed P, B halves every wave speed
    Ui4, Bi4 = _uniform_groups(1, N, ng, 4.0, (0.0, 0.0, 0.0), 0.6, (1.0, np.sqrt(2.0), 0.5))
    _, s4 = oracle.dt_reduce(cfg, Ui4, Bi4, ng, dh, cfl)
    assert abs(s4 - 0.5 * CFZ) < 1e-15


def test_dt_reads_interior_cells_only_and_every_group(oracle):
    N, ng, dh, cfl = 8, 3, 0.1, 0.3
    T = N + 2 * ng
    Ui, Bi = _uniform_groups(3, N, ng, 1.0, (0.0, 0.0, 0.0), 0.6, (1.0, np.sqrt(2.0), 0.5))
    cfg = oracle.make_config(N=N, g=3)
    U5 = Ui.reshape(3, 5, T, T, T).copy()
    e_moving = lambda vx: 0.6 / (G - 1) + 0.5 * vx * vx + 0.5 * 3.25
    # a fast cell in the ghost zone of group 0 must not count
    U5[0, 1, 1, 5, 5] = 50.0; U5[0, 4, 1, 5, 5] = e_moving(50.0)
    _, s = oracle.dt_reduce(cfg, U5.reshape(3, -1), Bi, ng, dh, cfl)
    assert abs(s - CFZ) < 1e-15
    # a fast interior cell of the LAST group, at the last interior index, must
    k = ng + N - 1
    U5[2, 1, k, k, k] = -3.0; U5[2, 4, k, k, k] = e_moving(3.0)
    _, s = oracle.dt_reduce(cfg, U5.reshape(3, -1), Bi, ng, dh, cfl)
    assert abs(s - 5.0) < 1e-14
    # the cell-centred field is the mean of the two faces (Eq. 5): doubling ONE x-face of one interior cell pair
    Bx = Bi[:, :T * T * (T + 1)].reshape(3, T, T, T + 1).copy()
    Bx[1, 5, 5, 6] = 3.0                        # cells (i=5) and (i=6) of row (5,5) now have Bc_x = 2
    B2 = Bi.copy(); B2[:, :T * T * (T + 1)] = Bx.reshape(3, -1)
    U5b = Ui.reshape(3, 5, T, T, T).copy()
    # keep P = 0.6 in those two cells: e = P/(g-1) + (Bc^2)/2 with Bc = (2, sqrt2, 1/2)
    for i in (5, 6):
        U5b[1, 4, 5, 5, i] = 0.6 / (G - 1) + 0.5 * (4.0 + 2.0 + 0.25)
    _, s = oracle.dt_reduce(cfg, U5b.reshape(3, -1), B2, ng, dh, cfl)
    # |B|^2 = 6.25, a^2 = 1; the largest speed is again along z (B_n^2 = 1/4): c_f^2 = (7.25 + sqrt(7.25^2 - 1))/2
    assert abs(s - np.sqrt((7.25 + np.sqrt(7.25 ** 2 - 1.0)) / 2.0)) < 1e-14
