"""P3 / P4 / P11 -- oracle Poisson + E (Eq. 1-2; Thomas, L142) against closed forms
and a dense numpy solve.  Wall-node E uses the half-cell Gauss law (R7).
O.solve_field() runs the oracle's field_solve() itself (the function the cycle executes), so a
wrong sign or index in its wall-node terms fails the closed forms below."""
import numpy as np
import pytest

from oracle import oracle as O
from helpers import params, load


@pytest.mark.parametrize("Nc", [2, 3, 8, 129, 1024])
def test_uniform_rho_closed_form(Nc):
    c = 0.75
    rho = np.full(Nc + 1, c)
    rho[0] = rho[-1] = c / 2          # raw wall-node sums of a uniform plasma
    phi, E = O.solve_field(Nc, 0, rho)
    j = np.arange(Nc + 1)
    assert np.allclose(phi, c * j * (Nc - j) / 2, rtol=1e-12, atol=1e-12 * Nc * Nc)
    assert np.allclose(E, c * (j - Nc / 2), rtol=1e-11, atol=1e-11 * Nc)


@pytest.mark.parametrize("Nc,m", [(16, 1), (64, 3), (257, 5)])
def test_sine_rho_bounded(Nc, m):
    j = np.arange(Nc + 1)
    rho = 2.5 * np.sin(np.pi * m * j / Nc)
    phi, E = O.solve_field(Nc, 0, rho)
    lam = 4 * np.sin(np.pi * m / (2 * Nc)) ** 2
    assert np.allclose(phi, rho / lam, rtol=1e-10, atol=1e-10 * np.abs(phi).max())
    ref = (np.roll(rho, 1) - np.roll(rho, -1))[1:-1] / (2 * lam)
    assert np.allclose(E[1:-1], ref, rtol=1e-9, atol=1e-10 * np.abs(E).max())


def test_laplace_and_superposition():
    Nc, V = 40, 123.0
    phi, E = O.solve_field(Nc, 0, np.zeros(Nc + 1), phi0=V, phiN=-7.0)
    j = np.arange(Nc + 1)
    assert np.allclose(phi, V + (-7.0 - V) * j / Nc, rtol=1e-12)
    assert np.allclose(E, (V + 7.0) / Nc, rtol=1e-11)          # P11: uniform E incl. walls
    rng = np.random.default_rng(0)
    r1, r2 = rng.normal(size=Nc + 1), rng.normal(size=Nc + 1)
    p1, E1 = O.solve_field(Nc, 0, r1, 1.0, 2.0)
    p2, E2 = O.solve_field(Nc, 0, r2, 3.0, -1.0)
    p3, E3 = O.solve_field(Nc, 0, r1 + r2, 4.0, 1.0)
    assert np.allclose(p1 + p2, p3, atol=1e-10) and np.allclose(E1 + E2, E3, atol=1e-10)


@pytest.mark.parametrize("Nc", [2, 5, 33, 64])
def test_thomas_vs_dense(Nc):
    rng = np.random.default_rng(Nc)
    rho = rng.normal(size=Nc + 1)
    phi0, phiN = 0.3, -1.1
    phi, E = O.solve_field(Nc, 0, rho, phi0, phiN)
    n = Nc - 1
    A = np.zeros((n, n))
    b = -rho[1:Nc].copy()
    for k in range(n):
        A[k, k] = -2
        if k > 0:
            A[k, k - 1] = 1
        if k < n - 1:
            A[k, k + 1] = 1
    b[0] -= phi0
    b[-1] -= phiN
    ref = np.linalg.solve(A, b) if n > 0 else np.zeros(0)
    assert np.allclose(phi[1:Nc], ref, atol=1e-11)
    assert np.isclose(E[0], (phi0 - phi[1]) - rho[0]) and np.isclose(E[Nc], (phi[Nc - 1] - phiN) + rho[Nc])


@pytest.mark.parametrize("Nc,m", [(8, 1), (64, 2), (512, 1)])
def test_periodic_sine(Nc, m):
    k = 2 * np.pi * m / Nc
    j = np.arange(Nc)
    a = 1.7
    rho = a * np.sin(k * j)
    lam = 4 * np.sin(k / 2) ** 2
    phi, E = O.solve_field(Nc, 1, rho)
    assert np.allclose(phi, rho / lam, atol=1e-9 * a / lam)
    assert np.allclose(E, -a * np.cos(k * j) * np.sin(k) / lam, atol=1e-9 * a / lam)
    phi2, E2 = O.solve_field(Nc, 1, rho + 5.0)     # neutralising mean is removed: gauge / offset free
    assert np.allclose(E, E2, atol=1e-9 * a / lam) and abs(phi2.mean()) < 1e-9 * a / lam


def test_rf_drive_no_charge_uniform_E():
    # P11 through the full cycle: no particles => E = V0 sin(omega (n+1)) / N_c at every node
    p = params(2, n_cells=16, ppc=1)
    o = O.Oracle(p)
    z = np.zeros(0, dtype=np.float32)
    load(o, [(z, z, z, z), (z, z, z, z)])
    for n in range(1, 6):
        o.step(1)
        rho, phi, E = o.get_rho_phi_E()
        assert not rho.any()
        assert np.allclose(E, p["V0_norm"] * np.sin(p["omega_dt"] * n) / 16, rtol=1e-12)


@pytest.mark.parametrize("Nc,f", [(8, 0.5), (64, 0.5), (33, 0.25)])
def test_uniform_plasma_through_the_full_cycle(Nc, f):
    """P3 through the full Oracle (load -> sort -> deposit -> field_solve): one ion per cell at the
    same offset f gives rho_j = 1 at interior nodes and the raw wall sums 1 - f and f.  For f = 1/2
    that is the uniform plasma with half-volume wall nodes: phi_j = j (N_c - j) / 2 and
    E_j = j - N_c / 2 at EVERY node including the walls (Eq. 1-2; R7).  For
    f != 1/2 the interior is the same parabola shifted by the wall-charge asymmetry; the wall
    fields follow from Gauss's law over the whole gap: E_N - E_0 = total charge = N_c."""
    p = params(2, n_cells=Nc, ppc=1, mcc=False, gamma=0.0)
    p["V0_norm"] = 0.0
    o = O.Oracle(p)
    z = np.zeros(0, np.float32)
    xi = (np.arange(Nc) + f).astype(np.float32)
    load(o, [(z, z, z, z), (xi, 0 * xi, 0 * xi, 0 * xi)])
    rho, phi, E = o.get_rho_phi_E()
    want = np.ones(Nc + 1)
    want[0], want[-1] = 1 - f, f
    assert np.array_equal(rho, want)
    j = np.arange(Nc + 1)
    assert np.isclose(E[-1] - E[0], Nc, rtol=1e-12)                  # Gauss over the gap
    assert np.allclose(np.diff(E)[1:-1], 1.0, rtol=1e-10)              # dE/dx = rho in the interior
    if f == 0.5:
        assert np.allclose(phi, j * (Nc - j) / 2, rtol=1e-12, atol=1e-12 * Nc * Nc)
        assert np.allclose(E, j - Nc / 2, rtol=1e-11, atol=1e-11 * Nc)
    else:
        # interior Poisson residual and the half-cell wall law, written out from Eq. 1-2
        assert np.allclose(phi[:-2] - 2 * phi[1:-1] + phi[2:], -rho[1:-1], atol=1e-10 * Nc)
        assert np.isclose(E[0], (phi[0] - phi[1]) - (1 - f), rtol=1e-12, atol=1e-12)
        assert np.isclose(E[-1], (phi[-2] - phi[-1]) + f, rtol=1e-12, atol=1e-12)
        # a wall-sign error would break the symmetry E_j(f) + E_{N-j}(1-f) = 0
    # mirror symmetry: reflecting the plasma (f -> 1 - f) reflects and negates E
    o2 = O.Oracle(p)
    xi2 = (np.arange(Nc) + (1 - f)).astype(np.float32)
    load(o2, [(z, z, z, z), (xi2, 0 * xi2, 0 * xi2, 0 * xi2)])
    _, phi2, E2 = o2.get_rho_phi_E()
    assert np.allclose(E2, -E[::-1], rtol=1e-11, atol=1e-11 * Nc)
    assert np.allclose(phi2, phi[::-1], rtol=1e-11, atol=1e-11 * Nc * Nc)


def test_wall_field_signs_single_sheet():
    """one positive charge sheet at node m between grounded walls (closed form of the discrete
    Green's function): phi_j = j (N - m) / N for j <= m, m (N - j) / N beyond; E is piecewise
    constant: -(N - m) / N left of the sheet and +m / N right of it, INCLUDING the wall nodes
    (rho_0 = rho_N = 0 there).  Pins the sign convention E = -dphi/dx at both walls."""
    N, m = 20, 7
    rho = np.zeros(N + 1)
    rho[m] = 1.0
    phi, E = O.solve_field(N, 0, rho)
    j = np.arange(N + 1)
    assert np.allclose(phi, np.where(j <= m, j * (N - m) / N, m * (N - j) / N), atol=1e-13)
    assert np.isclose(E[0], -(N - m) / N) and np.isclose(E[N], m / N)
    assert np.allclose(E[1:m], -(N - m) / N) and np.allclose(E[m + 1:N], m / N)
    # charge ON a wall node: the wall-node term of the half-cell law carries it (R7)
    rho = np.zeros(N + 1)
    rho[0] = 2.0
    phi, E = O.solve_field(N, 0, rho)
    assert not phi.any() and np.isclose(E[0], -2.0) and not E[1:].any()
    rho = np.zeros(N + 1)
    rho[N] = 3.0
    phi, E = O.solve_field(N, 0, rho)
    assert not phi.any() and np.isclose(E[N], 3.0) and not E[:N].any()
