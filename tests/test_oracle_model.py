"""Pins of the oracle's model step Phi, its TLM and its adjoint.

Every expected value here comes from mathematics outside the oracle: exact fixed points,
closed-form amplification matrices of the linearised scheme on a cylinder (cos_clamp = 1 makes
every metric factor 1, so rows decouple and Fourier / cosine modes are exact eigenmodes), the
textbook gravity-wave speed sqrt(g h0), the order of accuracy of centred differences, the
definition of a derivative (Taylor remainder) and the definition of an adjoint (PAPER.md:91
eq (3)).  A dropped term, a wrong sign or a swapped E/W or N/S index fails at least one.
"""
import numpy as np
import pytest

from oracle import Oracle
from paper_2205_06649_b200 import synth

G, H0, A_E, OM = synth.GRAVITY, synth.H0, synth.RADIUS, synth.OMEGA


def cylinder(nlon, nlat, dt, **kw):
    args = dict(cos_clamp=1.0, diffusion=0.0)
    args.update(kw)
    return Oracle(nlon, nlat, dt, 8, **args)


def test_row_tables_closed_form():
    o = Oracle(36, 18, 600.0, 4)
    t = o.row_tables()
    th = -np.pi / 2 + (np.arange(18) + 0.5) * np.pi / 18
    mc = np.maximum(np.cos(th), np.cos(np.deg2rad(50.0)))
    assert np.allclose(t["mc"], mc, rtol=1e-15)
    assert np.allclose(t["f"], 2 * OM * np.sin(th), rtol=1e-14)
    assert np.allclose(t["t"], np.sin(th) / (A_E * mc), rtol=1e-14)
    assert np.allclose(t["cz"], 1 / (2 * A_E * (2 * np.pi / 36) * mc), rtol=1e-14)
    assert np.isclose(t["cm"], 1 / (2 * A_E * np.pi / 18), rtol=1e-14)
    assert t["rp"][-1] == 1.0 and t["rm"][0] == 1.0
    assert np.allclose(t["rp"][:-1], mc[1:] / mc[:-1], rtol=1e-15)
    assert np.allclose(t["rm"][1:], mc[:-1] / mc[1:], rtol=1e-15)


def test_rest_state_is_exact_fixed_point():
    o = Oracle(36, 18, 600.0, 4)
    Z = np.zeros((3, 18, 36)); Z[0] = H0
    assert np.array_equal(o.step(Z), Z)


def test_zonal_gravity_wave_closed_form_and_speed():
    """Omega = 0, kappa = 0, cylinder: mode e^{ik lambda} of (eta,u) is advanced by
    [[1, -i s h0], [-i s g, 1 - s^2 g h0]], s = 2 dt cz sin(k dlambda) (forward-backward);
    an eastward-travelling wave moves at ~ sqrt(g h0)."""
    nlon, nlat, dt, k, n = 72, 6, 300.0, 3, 12
    o = cylinder(nlon, nlat, dt, omega=0.0)
    cz = o.row_tables()["cz"][0]
    lam = np.arange(nlon) * 2 * np.pi / nlon
    eps = 1e-3
    Z = np.zeros((3, nlat, nlon))
    Z[0] = H0 + eps * np.cos(k * lam)[None, :]
    Z[1] = eps * np.sqrt(G / H0) * np.cos(k * lam)[None, :]       # eastward-travelling
    s = 2 * dt * cz * np.sin(k * 2 * np.pi / nlon)
    M = np.array([[1, -1j * s * H0], [-1j * s * G, 1 - s * s * G * H0]])
    amp = np.linalg.matrix_power(M, n) @ np.array([eps, eps * np.sqrt(G / H0)], dtype=complex)
    for _ in range(n):
        Z = o.step(Z)
    eta = np.real(amp[0] * np.exp(1j * k * lam))
    u = np.real(amp[1] * np.exp(1j * k * lam))
    assert np.abs(Z[0] - H0 - eta[None, :]).max() < 1e-5 * eps
    assert np.abs(Z[1] - u[None, :]).max() < 1e-5 * eps * np.sqrt(G / H0)
    assert np.abs(Z[2]).max() < 1e-6 * eps
    # textbook speed: the crest phase moved east by k*c*T/a (3 % numerical-dispersion allowance)
    phase = -np.angle(amp[0])
    assert phase == pytest.approx(k * np.sqrt(G * H0) * n * dt / A_E, rel=0.03)


def test_meridional_standing_wave_closed_form():
    """h = cos(alpha (j+1/2)), v = sin(alpha (j+1/2)) are exact eigenmodes of centred
    differences with the reflective pole walls (ghost row = edge row, v negated)."""
    nlon, nlat, dt, l, n = 8, 24, 300.0, 2, 15
    o = cylinder(nlon, nlat, dt, omega=0.0)
    cm = o.row_tables()["cm"]
    al = l * np.pi / nlat
    cj, sj = np.cos(al * (np.arange(nlat) + 0.5)), np.sin(al * (np.arange(nlat) + 0.5))
    eps = 1e-3
    Z = np.zeros((3, nlat, nlon)); Z[0] = H0 + eps * cj[:, None]
    s = 2 * dt * cm * np.sin(al)
    M = np.array([[1, -s * H0], [s * G, 1 - s * s * G * H0]])
    amp = np.linalg.matrix_power(M, n) @ np.array([eps, 0.0])
    for _ in range(n):
        Z = o.step(Z)
    assert np.abs(Z[0] - H0 - amp[0] * cj[:, None]).max() < 1e-5 * eps
    assert np.abs(Z[2] - amp[1] * sj[:, None]).max() < 1e-5 * eps * np.sqrt(G / H0)
    assert abs(amp[1]) > 0.1 * eps * np.sqrt(G / H0)          # the test is not vacuous


def test_inertial_oscillation_closed_form():
    """g = 0: a uniform wind rotates clockwise in the northern hemisphere; per row
    (u,v) <- [[1, a], [-a, 1 - a^2]] (u,v), a = dt f_j (forward-backward Coriolis)."""
    nlon, nlat, dt, n = 8, 12, 600.0, 20
    o = cylinder(nlon, nlat, dt, gravity=0.0)
    f = o.row_tables()["f"]
    eps = 1e-4
    Z = np.zeros((3, nlat, nlon)); Z[0] = H0; Z[1] = eps
    for _ in range(n):
        Z = o.step(Z)
    for j in range(2, nlat - 2):
        a = dt * f[j]
        uv = np.linalg.matrix_power(np.array([[1, a], [-a, 1 - a * a]]), n) @ np.array([eps, 0.0])
        assert np.abs(Z[1, j] - uv[0]).max() < 2e-6 * eps
        assert np.abs(Z[2, j] - uv[1]).max() < 2e-6 * eps
    assert Z[2, nlat - 3, 0] < 0 < Z[2, 2, 0]                  # clockwise north, anticlockwise south


@pytest.mark.parametrize("kappa", [0.0, 0.02])
def test_one_step_zonal_advection_diffusion_amplification(kappa):
    """Uniform zonal wind U: one step multiplies mode e^{ik lambda} of h by
    G = 1 - 2i dt cz U sin(k dl) + kappa (2 cos(k dl) - 2)  (FTCS advection + diffusion)."""
    nlon, nlat, dt, k, U, A = 48, 6, 300.0, 4, 12.0, 100.0
    o = cylinder(nlon, nlat, dt, omega=0.0, gravity=0.0, diffusion=kappa)
    cz = o.row_tables()["cz"][0]
    lam = np.arange(nlon) * 2 * np.pi / nlon
    Z = np.zeros((3, nlat, nlon)); Z[0] = H0 + A * np.cos(k * lam)[None, :]; Z[1] = U
    dl = k * 2 * np.pi / nlon
    Gf = 1 - 2j * dt * cz * U * np.sin(dl) + kappa * (2 * np.cos(dl) - 2)
    Z1 = o.step(Z)
    exp = H0 + A * np.real(Gf * np.exp(1j * k * lam))
    assert np.abs(Z1[0, 2:-2] - exp[None, :]).max() < 1e-9
    assert np.angle(Gf) < 0                                    # pattern moves downwind (east)


def test_one_step_meridional_advection_amplification():
    nlon, nlat, dt, l, V, A, kappa = 6, 32, 300.0, 3, 8.0, 100.0, 0.02
    o = cylinder(nlon, nlat, dt, omega=0.0, gravity=0.0, diffusion=kappa)
    cm = o.row_tables()["cm"]
    al = l * np.pi / nlat
    cj, sj = np.cos(al * (np.arange(nlat) + 0.5)), np.sin(al * (np.arange(nlat) + 0.5))
    Z = np.zeros((3, nlat, nlon)); Z[0] = H0 + A * cj[:, None]; Z[2] = V
    Z1 = o.step(Z)
    exp = H0 + A * (cj + 2 * dt * cm * V * np.sin(al) * sj + kappa * (2 * np.cos(al) - 2) * cj)
    assert np.abs(Z1[0, 3:-3] - exp[3:-3, None]).max() < 1e-9


def test_balanced_zonal_flow_drift_is_second_order():
    """u = u0 cos(theta), h = h0 - (a Omega u0 + u0^2/2) sin^2(theta)/g is a steady state of
    eq (60)-(62): one discrete step leaves h,u unchanged and drifts v by
    dt*O(dtheta^2), so the drift falls ~4x per grid halving (equatorward of the metric clamp)."""
    drift = []
    for nlat in (18, 36, 72):
        nlon = 2 * nlat
        o = Oracle(nlon, nlat, 60.0, 2, diffusion=0.0)
        th = -np.pi / 2 + (np.arange(nlat) + 0.5) * np.pi / nlat
        Z = np.zeros((3, nlat, nlon))
        Z[1] = (synth.U0 * np.cos(th))[:, None]
        Z[0] = (H0 - (A_E * OM * synth.U0 + synth.U0 ** 2 / 2) * np.sin(th) ** 2 / G)[:, None]
        Z1 = o.step(Z)
        rows = np.abs(th) < np.deg2rad(44.0)
        assert np.abs(Z1[0] - Z[0]).max() < 1e-9 and np.abs(Z1[1] - Z[1]).max() < 1e-12
        drift.append(np.abs(Z1[2][rows]).max() / 60.0)
    assert 3.5 < drift[0] / drift[1] < 4.6 and 3.5 < drift[1] / drift[2] < 4.6
    # and the Coriolis / pressure-gradient terms it balances are each ~1e-3 m/s^2, i.e. the
    # residual is a small difference of large terms, not two zeros
    assert drift[2] < 1e-3 * 2 * OM * synth.U0


@pytest.fixture(scope="module")
def cfg0():
    w = synth.CONFIGS[0]
    return Oracle(w.nlon, w.nlat, w.dt, w.nsteps), synth.background(
        w, synth.truth_initial(w), synth.sigmas(synth.truth_initial(w))[0])


def test_tlm_taylor_remainder(cfg0):
    o, Z = cfg0
    d = synth.random_fields(Z.shape, 11) * np.array([10.0, 1.0, 1.0])[:, None, None]
    base, lin = o.step(Z), o.step_tlm(Z, d)
    rem = [np.abs(o.step(Z + e * d) - base - e * lin).max() / e ** 2 for e in (1e-1, 1e-2, 1e-3)]
    assert max(rem) < 3 * min(rem) and min(rem) > 0          # O(eps^2), constant bounded
    assert np.abs(lin).max() > 1.0


def test_step_adjoint_dot_product_identity(cfg0):
    """PAPER.md:91 eq (3): <y, A x> = <A^T y, x> to 1e-12 relative."""
    o, Z = cfg0
    for seed in range(3):
        d = synth.random_fields(Z.shape, 20 + seed)
        y = synth.random_fields(Z.shape, 40 + seed)
        a, b = np.vdot(o.step_tlm(Z, d), y), np.vdot(d, o.step_adj(Z, y))
        assert abs(a - b) <= 1e-12 * abs(a)


def test_window_adjoint_is_reverse_product(cfg0):
    """PAPER.md:98 eq (4): (M^{0,n})^T = (M^{0,1})^T ... applied in reverse order."""
    o, Z = cfg0
    d = synth.random_fields(Z.shape, 5); y = synth.random_fields(Z.shape, 6)
    traj = [Z]
    for _ in range(4):
        traj.append(o.step(traj[-1]))
    t = d
    for n in range(4):
        t = o.step_tlm(traj[n], t)
    a = y
    for n in reversed(range(4)):
        a = o.step_adj(traj[n], a)
    assert abs(np.vdot(t, y) - np.vdot(d, a)) <= 1e-12 * abs(np.vdot(t, y))
